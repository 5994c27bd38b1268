// Host side of libmwf.so: the C ABI of include/mwf.h -- device store, list-reuse driver (SURVEY.md
// section 8(a) rows a1, a2, a5, a6, a7) and the launches of the kernels in this directory.
#include <algorithm>
#include <chrono>
#include <cstdlib>
#include <climits>
#include <cstdio>
#include <cstring>
#include <new>
#include <numeric>

#include "mwf_internal.h"
#include "scan_sort.cuh"

using namespace mwf;

struct mwf_ctx {
    mwf_params p{};
    int n_sm = 0, ctas_per_sm = 0;
    int64_t l2_bytes = 0;
    char* arena = nullptr;
    int64_t arena_bytes = 0;
    bool own_arena = false;
    // carved device arrays
    float4* store = nullptr;      // [max_ptcl + max_cell + 1]
    float4* store_next = nullptr; // same size: the shadow store of the pipelined host loop (mwf_set_particles_next / mwf_swap_store)
    int64_t next_count = 0;       // particles written into the shadow store since the last swap
    std::vector<cudaStream_t> next_streams;  // streams those uploads went to
    float4* accp = nullptr;       // [max_ptcl]
    float4* vel = nullptr;        // [max_ptcl] (vx, vy, vz, unused): device-resident integration
    mwf_cell* cells = nullptr;    // [max_cell]
    int32_t* parent = nullptr;    // [max_cell]
    int32_t* arrive = nullptr;    // [max_cell]
    double4* mom64 = nullptr;     // [max_cell]
    int2* cell_lr = nullptr;      // [max_cell] range of leaf ranks of every cell (scan variant of the refresh)
    double4* leaf_P = nullptr;    // [max_cell + 1] leaves' moments in rank order, scanned in place every refresh
    double4* leaf_toff = nullptr; // [tiles] scanned tile totals
    int64_t n_leaf_cells = 0;
    int32_t* grp_first = nullptr; // [max_group]
    int32_t* grp_n = nullptr;     // [max_group]
    uint8_t* grp_self = nullptr;  // [max_group]
    int64_t* list_off = nullptr;  // [max_group + 1]
    int64_t* st_epj_off = nullptr, *st_spj_off = nullptr;  // [max_group + 1] staging
    int32_t* st_ids = nullptr;    // [max_entry] staging of the uploaded ids
    int32_t* list = nullptr;      // [max_entry + TILE_J * max_group] merged, padded
    WorkItem* items = nullptr;    // [max_items]
    int32_t* order_full = nullptr, *order_split = nullptr;  // [max_items]
    unsigned int* counters = nullptr;  // [N_COUNTER]
    unsigned int* err = nullptr;
    int64_t max_items = 0;
    // state
    int64_t n_ptcl = 0, n_cell = 0, n_group = 0, n_items = 0, ptcl_hi = 0, padded_entries = 0;
    bool have_tree = false, have_lists = false, lists_for_reuse = false, mono_fresh = false;
    BuildBuffers bb{};       // device-side construction step (NEXT-2)
    int64_t walk_warps_n = 0;
    bool built_on_device = false;
    int64_t build_e_epj = 0, build_e_spj = 0;
    int32_t build_n_level = 0;
    bool acc_full = false;   // every group has been dispatched since the positions last changed
    int64_t vel_hi = 0;      // velocities [0, vel_hi) have been uploaded
    std::vector<int64_t> h_item_off, h_inter, h_split;  // per group prefix of items / interactions; split group bounds
    std::vector<int32_t> h_grp_first, h_grp_n;
    std::vector<WorkItem> h_items;   // kept for the per-tag schedule, which is made on first use
    std::vector<int64_t> h_cost;
    bool split_ready = false;
    int64_t groups_outstanding = 0;  // MAKE_LIST: groups dispatched and not yet retrieved
    int64_t groups_dispatched = 0;
    // streams and events
    cudaStream_t tag_stream[MWF_MAX_TAG]{};
    bool tag_own[MWF_MAX_TAG]{};
    bool tag_inflight[MWF_MAX_TAG]{};
    cudaEvent_t ev_tag[MWF_MAX_TAG]{}, ev_k0[MWF_MAX_TAG]{}, ev_k1[MWF_MAX_TAG]{};
    bool tag_timed[MWF_MAX_TAG]{};
    cudaEvent_t ev_store{};
    cudaEvent_t ev_next{};
    bool store_event_valid = false;
    std::vector<std::pair<int64_t, int64_t>> tag_ranges[MWF_MAX_TAG];  // particle ranges awaiting retrieve
    std::vector<int64_t> tag_groups;                                   // groups awaiting retrieve per tag
    // method G1 (data lists, NEXT-3): per-tag staging of j records and their offsets, cudaMalloc'ed on demand
    float4* data_buf[MWF_MAX_TAG]{};
    int64_t* data_off[MWF_MAX_TAG]{};
    int64_t data_cap = 0;
    // quadrupole SPJ (NEXT-3): cudaMalloc'ed when mwf_set_spj_order(2) is first called
    int spj_order = 1;
    double* quad64 = nullptr;   // [6 * max_cell]
    float4* quad = nullptr;     // [2 * max_cell]
    int quad_ctas_per_sm = 0;
    cudaEvent_t ev_kq[MWF_MAX_TAG]{};
    bool tag_quad[MWF_MAX_TAG]{};
    // short-range workload (NEXT-4): per-particle SPH record, cudaMalloc'ed when mwf_set_sph() is first called
    float4* sph = nullptr;      // [max_ptcl] (h, u, rho, P/rho^2)
    int64_t sph_hi = 0;         // records [0, sph_hi) have been uploaded
    int sph_ctas_per_sm[2] = {0, 0};
    int tag_kind[MWF_MAX_TAG]{};  // what the tag's pending results are: 0 = acc/pot (or hydro acc), 1 = SPH records
    uint32_t counter_seq = 0;
    int64_t n_launch = 0, n_inter = 0;
    std::string cuda_err;
};

namespace {

constexpr int N_COUNTER = 1024;

// MWF_TRACE=1 in the environment: wall-clock phase times of the construction step on stderr
bool trace_on() {
    static const bool on = [] { const char* e = std::getenv("MWF_TRACE"); return e && e[0] && e[0] != '0'; }();
    return on;
}
struct PhaseTimer {
    std::chrono::steady_clock::time_point t0 = std::chrono::steady_clock::now();
    void lap(const char* what) {
        if (!trace_on()) return;
        const auto t1 = std::chrono::steady_clock::now();
        fprintf(stderr, "[mwf trace] %-28s %8.3f ms\n", what, std::chrono::duration<double, std::milli>(t1 - t0).count());
        t0 = t1;
    }
};

int cuda_fail(mwf_ctx* c, cudaError_t e, const char* what) {
    if (c) {
        char buf[256];
        snprintf(buf, sizeof buf, "%s: %s", what, cudaGetErrorString(e));
        c->cuda_err = buf;
    }
    return MWF_ECUDA;
}
#define CU(c, call)                                                   \
    do {                                                              \
        cudaError_t e__ = (call);                                     \
        if (e__ != cudaSuccess) return cuda_fail((c), e__, #call);    \
    } while (0)

inline int64_t up(int64_t x, int64_t a) { return (x + a - 1) / a * a; }

struct Layout {
    int64_t off[48];
    int n = 0;
    int64_t total = 0;
    int64_t add(int64_t bytes) {
        off[n] = total;
        total += up(bytes, 256);
        return off[n++];
    }
};

int64_t max_items_of(const mwf_params& p) { return p.max_ptcl / CHUNK_I + 5 * p.max_group + 8; }

Layout make_layout(const mwf_params& p) {
    Layout L;
    const int64_t mi = max_items_of(p);
    L.add((p.max_ptcl + p.max_cell + 1) * 16);          // 0 store
    L.add(p.max_ptcl * 16);                             // 1 accp
    L.add(p.max_cell * 16);                             // 2 cells
    L.add(p.max_cell * 4);                              // 3 parent
    L.add(p.max_cell * 4);                              // 4 arrive
    L.add(p.max_cell * 32);                             // 5 mom64
    L.add(p.max_group * 4);                             // 6 grp_first
    L.add(p.max_group * 4);                             // 7 grp_n
    L.add(p.max_group);                                 // 8 grp_self
    L.add((p.max_group + 1) * 8);                       // 9 list_off
    L.add((p.max_group + 1) * 8);                       // 10 st_epj_off
    L.add((p.max_group + 1) * 8);                       // 11 st_spj_off
    L.add(p.max_entry * 4);                             // 12 st_ids
    L.add((p.max_entry + TILE_J * p.max_group) * 4);    // 13 list
    L.add(mi * (int64_t)sizeof(WorkItem));              // 14 items
    L.add(mi * 4);                                      // 15 order_full
    L.add(mi * 4);                                      // 16 order_split
    L.add(N_COUNTER * 4);                               // 17 counters
    L.add(256);                                         // 18 err
    L.add(p.max_ptcl * 16);                             // 19 vel
    // device-side construction step (NEXT-2)
    const int64_t nsb = sort_blocks(p.max_ptcl);
    const int64_t scan_n = std::max<int64_t>(std::max<int64_t>(256 * nsb + 1, p.max_ptcl + 2), p.max_cell + 2);
    L.add(p.max_ptcl * 8);                              // 20 key_a
    L.add(p.max_ptcl * 8);                              // 21 key_b
    L.add(p.max_ptcl * 4);                              // 22 idx_a (the permutation after a build)
    L.add(p.max_ptcl * 4);                              // 23 idx_b
    L.add((256 * nsb + 1) * 4);                         // 24 hist
    L.add(scan_scratch_elems(scan_n) * 4);              // 25 scan_scratch (int32)
    L.add(scan_scratch_elems(p.max_group + 2) * 8);     // 26 scan_scratch64
    L.add(148 * 4 * 6 * 4);                             // 27 bbox_part
    L.add(8 * 8);                                       // 28 root
    L.add(p.max_cell * 32);                             // 29 geom
    L.add((p.max_cell + 2) * 4);                        // 30 level_cnt
    L.add((p.max_ptcl + 2) * 4);                        // 31 mark
    L.add(p.max_group * 4);                             // 32 grp_cell
    L.add(p.max_group * 24);                            // 33 grp_box
    L.add(p.max_group * 4);                             // 34 n_epj
    L.add(p.max_group * 4);                             // 35 n_spj
    L.add(walk_warps(p.max_group) * WALK_STACK * 4);    // 36 walk_stacks
    L.add(256);                                         // 37 walk_counter
    L.add((p.max_cell + 2) * 32);                       // 38 level_bounds (8 octant ends per cell of the level being split)
    L.add(p.max_cell * 8);                              // 39 cell_lr
    L.add((p.max_cell + 1) * 32);                       // 40 leaf_P
    L.add((scan4_tiles(p.max_cell) + 1) * 32);          // 41 leaf_toff
    L.add((p.max_ptcl + p.max_cell + 1) * 16);          // 42 store_next
    return L;
}

bool params_ok(const mwf_params* p) {
    if (!p) return false;
    if (!(p->eps > 0.f) || !(p->eps * p->eps >= 1.17549435e-38f)) return false;
    if (!(p->G == p->G)) return false;
    if (p->max_ptcl < 1 || p->max_cell < 1 || p->max_group < 1 || p->max_entry < 1) return false;
    if (p->max_ptcl + p->max_cell + 1 > 0x7fffffffLL) return false;  // 32-bit list indices
    if (p->n_tag < 1 || p->n_tag > MWF_MAX_TAG) return false;
    if (p->device < 0) return false;
    return true;
}

// Every operation that writes the store / tree / lists first waits for the force kernels that read them.
int before_store_op(mwf_ctx* c, cudaStream_t s) {
    for (int t = 0; t < c->p.n_tag; ++t)
        if (c->tag_inflight[t]) CU(c, cudaStreamWaitEvent(s, c->ev_tag[t], 0));
    if (c->store_event_valid) CU(c, cudaStreamWaitEvent(s, c->ev_store, 0));
    return MWF_OK;
}
int after_store_op(mwf_ctx* c, cudaStream_t s) {
    CU(c, cudaEventRecord(c->ev_store, s));
    c->store_event_valid = true;
    return MWF_OK;
}

int read_err_word(mwf_ctx* c, cudaStream_t s, unsigned int* out) {
    CU(c, cudaMemcpyAsync(out, c->err, sizeof(unsigned int), cudaMemcpyDeviceToHost, s));
    CU(c, cudaStreamSynchronize(s));
    return MWF_OK;
}

void drop_lists(mwf_ctx* c) {
    c->have_lists = false;
    c->lists_for_reuse = false;
    c->n_group = 0;
    c->n_items = 0;
    c->groups_dispatched = 0;
    c->acc_full = false;
}

// Work order of items [b, e) of `order`: longest first (so the tail of the launch is made of short items),
// except that the NARROW items (width <= 8: few j-pairs per staged tile, so they wait on the gathers rather
// than on the FP32 pipe) are spread evenly over the first 7/8 of the schedule, where the wide items of the
// other warps of the SM keep the pipe busy meanwhile.
// Stable LSD radix sort (11-bit digits) of item indices by DESCENDING cost: O(n), ties keep item order.
void sort_longest_first(std::vector<int32_t>& v, const std::vector<int64_t>& cost, std::vector<int32_t>& tmp) {
    const size_t n = v.size();
    if (n < 2) return;
    int64_t cmax = 0;
    for (int32_t it : v) cmax = std::max(cmax, cost[(size_t)it]);
    tmp.resize(n);
    for (int shift = 0; shift < 63 && (cmax >> shift) > 0; shift += 11) {
        size_t count[2049] = {0};
        for (int32_t it : v) ++count[(size_t)(((cmax - cost[(size_t)it]) >> shift) & 2047) + 1];
        for (int d = 0; d < 2048; ++d) count[d + 1] += count[d];
        for (int32_t it : v) tmp[count[(size_t)(((cmax - cost[(size_t)it]) >> shift) & 2047)]++] = it;
        v.swap(tmp);
    }
}

void schedule_items(std::vector<int32_t>& order, int64_t b, int64_t e, const std::vector<WorkItem>& items, const std::vector<int64_t>& cost) {
    std::vector<int32_t> wide, narrow, tmp;
    wide.reserve((size_t)(e - b));
    for (int64_t k = b; k < e; ++k) {
        const int32_t it = order[(size_t)k];
        (items[(size_t)it].width > 8 ? wide : narrow).push_back(it);
    }
    sort_longest_first(wide, cost, tmp);
    sort_longest_first(narrow, cost, tmp);
    const size_t nw = wide.size(), nn = narrow.size();
    const size_t span = nw - nw / 8;  // narrow items go between the first `span` wide items
    size_t iw = 0, in = 0;
    int64_t k = b;
    while (iw < nw || in < nn) {
        // keep in / nn ~ iw / span
        const bool take_narrow = in < nn && (iw >= nw || (span > 0 ? in * span <= iw * nn : true) || iw >= span);
        order[(size_t)k++] = take_narrow ? narrow[in++] : wide[iw++];
    }
}

// MWF_REFRESH=climb in the environment: the bottom-up climb also for monopoles (A/B switch for the scan variant)
bool use_scan_refresh() {
    static const bool on = [] { const char* e = std::getenv("MWF_REFRESH"); return !(e && e[0] == 'c'); }();
    return on;
}

// Host-side work plan of one set of lists: per-group list offsets (padded to tiles), work items, the two
// schedules, and the per-group prefix sums the dispatcher needs.  Used by mwf_set_lists (lists from the host)
// and by mwf_build (lists made on the device; only their lengths come back).
struct Plan {
    std::vector<int64_t> list_off, item_off, inter, split;
    std::vector<WorkItem> items;
    std::vector<int64_t> cost;
    std::vector<int32_t> order_full;
};

int make_plan(mwf_ctx* c, int64_t n_group, const int32_t* grp_first, const int32_t* grp_n, const int64_t* n_list_of, Plan& pl) {
    pl.list_off.assign((size_t)n_group + 1, 0);
    pl.item_off.assign((size_t)n_group + 1, 0);
    pl.inter.assign((size_t)n_group + 1, 0);
    std::vector<WorkItem>& items = pl.items;
    std::vector<int64_t>& cost = pl.cost;
    items.reserve((size_t)(c->n_ptcl / CHUNK_I + 3 * n_group));
    for (int64_t g = 0; g < n_group; ++g) {
        const int64_t gf = grp_first[g], gn = grp_n[g];
        if (gf < 0 || gn < 1 || gf + gn > c->n_ptcl) return MWF_ERANGE;
        const int64_t n_list = n_list_of[g];
        const int64_t n_tiles = (n_list + TILE_J - 1) / TILE_J;
        pl.list_off[(size_t)g + 1] = pl.list_off[(size_t)g] + n_tiles * TILE_J;
        pl.inter[(size_t)g + 1] = pl.inter[(size_t)g] + gn * n_list;
        // Cut the group into items: whole 64-particle items, then power-of-two pieces of the remainder
        // padded to a multiple of q; q is the quantum whose modelled cost is lowest (a coarser quantum
        // wastes lanes, a finer one re-stages the list for one more narrow item).
        const int64_t n_full = gn / CHUNK_I, rem = gn % CHUNK_I;
        int64_t best_q = CHUNK_I, best_cost = INT64_MAX;
        for (int64_t q = 2 * MIN_WIDTH; q <= CHUNK_I && rem > 0; q *= 2) {
            const int64_t padded = (rem + q - 1) / q * q;
            int64_t cst = 0;
            for (int64_t piece = CHUNK_I; piece >= 2 * MIN_WIDTH; piece /= 2)
                if (padded & piece) cst += item_cost_per_tile((int)(piece / 2));
            if (cst < best_cost) { best_cost = cst; best_q = q; }
        }
        int64_t done = 0;
        auto emit = [&](int64_t n_i, int width) {
            WorkItem it;
            it.i_first = (int32_t)(gf + done);
            it.n_i = (int32_t)n_i;
            it.group = (int32_t)g;
            it.width = width;
            done += n_i;
            items.push_back(it);
            cost.push_back(n_tiles * item_cost_per_tile(width));
        };
        for (int64_t k = 0; k < n_full; ++k) emit(CHUNK_I, CHUNK_I / 2);
        if (rem > 0) {
            const int64_t padded = (rem + best_q - 1) / best_q * best_q;
            for (int64_t piece = CHUNK_I; piece >= 2 * MIN_WIDTH; piece /= 2)
                if (padded & piece) emit(std::min(piece, gn - done), (int)(piece / 2));
        }
        pl.item_off[(size_t)g + 1] = (int64_t)items.size();
    }
    const int64_t n_items = (int64_t)items.size();
    if (n_items > c->max_items) return MWF_ENOMEM;
    // work schedule over everything (see schedule_items); the schedules inside the n_tag interaction-balanced group
    // ranges that mwf_calc_force_all uses for a host destination are made on first use (ensure_split_order)
    pl.order_full.resize((size_t)n_items);
    std::iota(pl.order_full.begin(), pl.order_full.end(), 0);
    // A store that does not fit the L2 is walked in SCHED_WINDOWS windows of consecutive (Morton-ordered) items of equal
    // modelled cost, each scheduled as above: the gathers of the items in flight then touch one stretch of the store at a
    // time (config 4, 171 MB store: DRAM traffic 6.7 -> 3.1 GB per launch at the same kernel time; a store that fits loses
    // 0.3-0.7 % to the less even mix of long and short items, so it keeps one window).
    const int64_t store_bytes = (c->n_ptcl + c->n_cell + 1) * (int64_t)sizeof(float4);
    const int n_win = store_bytes > c->l2_bytes ? SCHED_WINDOWS : 1;
    if (n_win <= 1) {
        schedule_items(pl.order_full, 0, n_items, items, cost);
    } else {
        int64_t tot = 0;
        for (int64_t k = 0; k < n_items; ++k) tot += cost[(size_t)k];
        int64_t b = 0, acc = 0;
        for (int w = 1; w <= n_win && b < n_items; ++w) {
            const int64_t want = tot / n_win * w;
            int64_t e = b;
            while (e < n_items && (acc < want || w == n_win)) acc += cost[(size_t)e++];
            schedule_items(pl.order_full, b, e, items, cost);
            b = e;
        }
    }
    pl.split.assign((size_t)c->p.n_tag + 1, 0);
    const int64_t total = pl.inter[(size_t)n_group];
    int64_t g = 0;
    for (int t = 1; t < c->p.n_tag; ++t) {
        const int64_t want = total / c->p.n_tag * t;
        while (g < n_group && pl.inter[(size_t)g] < want) ++g;
        pl.split[(size_t)t] = g;
    }
    pl.split[(size_t)c->p.n_tag] = n_group;
    return MWF_OK;
}

// Adopt a plan as the ctx's current lists (after the device side is in place).
void adopt_plan(mwf_ctx* c, Plan& pl, int64_t n_group, const int32_t* grp_first, const int32_t* grp_n, int mode) {
    c->h_item_off.swap(pl.item_off);
    c->h_inter.swap(pl.inter);
    c->h_split.swap(pl.split);
    c->h_items.swap(pl.items);
    c->h_cost.swap(pl.cost);
    c->split_ready = false;
    c->h_grp_first.assign(grp_first, grp_first + n_group);
    c->h_grp_n.assign(grp_n, grp_n + n_group);
    c->n_group = n_group;
    c->n_items = (int64_t)c->h_items.size();
    c->padded_entries = pl.list_off[(size_t)n_group];
    c->have_lists = true;
    c->lists_for_reuse = (mode == MWF_MAKE_LIST_FOR_REUSE);
    c->groups_dispatched = 0;
    c->groups_outstanding = 0;
}

// Per-tag schedules: made and uploaded the first time a dispatch covers exactly one of the balanced ranges.
int ensure_split_order(mwf_ctx* c, cudaStream_t s) {
    if (c->split_ready) return MWF_OK;
    std::vector<int32_t> order((size_t)c->n_items);
    std::iota(order.begin(), order.end(), 0);
    for (int t = 0; t < c->p.n_tag; ++t) {
        const int64_t b = c->h_item_off[(size_t)c->h_split[(size_t)t]], e = c->h_item_off[(size_t)c->h_split[(size_t)t + 1]];
        schedule_items(order, b, e, c->h_items, c->h_cost);
    }
    CU(c, cudaMemcpyAsync(c->order_split, order.data(), (size_t)c->n_items * 4, cudaMemcpyHostToDevice, s));
    CU(c, cudaStreamSynchronize(s));
    c->split_ready = true;
    return MWF_OK;
}

}  // namespace

extern "C" {

const char* mwf_strerror(int code) {
    switch (code) {
        case MWF_OK: return "ok";
        case MWF_EINVAL: return "invalid argument";
        case MWF_ESTATE: return "call out of order for the current list/monopole state";
        case MWF_ERANGE: return "index, range or offset out of bounds in the uploaded tree or lists";
        case MWF_ENOMEM: return "capacity exceeded";
        case MWF_ECUDA: return "CUDA error";
        default: return "unknown error code";
    }
}

const char* mwf_last_cuda_error(mwf_ctx* c) { return c ? c->cuda_err.c_str() : ""; }

int mwf_arena_bytes(const mwf_params* p, int64_t* bytes) {
    if (!params_ok(p) || !bytes) return MWF_EINVAL;
    *bytes = make_layout(*p).total;
    return MWF_OK;
}

int mwf_create(mwf_ctx** out, const mwf_params* p, void* arena, int64_t arena_bytes) {
    if (!out) return MWF_EINVAL;
    *out = nullptr;
    if (!params_ok(p)) return MWF_EINVAL;
    mwf_ctx* c = new (std::nothrow) mwf_ctx;
    if (!c) return MWF_ENOMEM;
    c->p = *p;
    cudaError_t e = cudaSetDevice(p->device);
    if (e != cudaSuccess) { delete c; return MWF_ECUDA; }
    cudaDeviceProp prop;
    e = cudaGetDeviceProperties(&prop, p->device);
    if (e != cudaSuccess) { delete c; return MWF_ECUDA; }
    if (prop.major != 10) {  // sm_100a code only: fail loudly, there is no fallback
        delete c;
        return MWF_ECUDA;
    }
    c->n_sm = prop.multiProcessorCount;
    c->l2_bytes = prop.l2CacheSize;
    c->ctas_per_sm = force_max_ctas_per_sm();
    if (c->ctas_per_sm < 1) { delete c; return MWF_ECUDA; }
    const Layout L = make_layout(*p);
    if (arena) {
        if (arena_bytes < L.total || (reinterpret_cast<uintptr_t>(arena) & 255)) { delete c; return MWF_ENOMEM; }
        c->arena = static_cast<char*>(arena);
    } else {
        void* m = nullptr;
        if (cudaMalloc(&m, (size_t)L.total) != cudaSuccess) { cudaGetLastError(); delete c; return MWF_ENOMEM; }
        c->arena = static_cast<char*>(m);
        c->own_arena = true;
    }
    c->arena_bytes = L.total;
    char* b = c->arena;
    c->store = (float4*)(b + L.off[0]);
    c->store_next = (float4*)(b + L.off[42]);
    c->accp = (float4*)(b + L.off[1]);
    c->cells = (mwf_cell*)(b + L.off[2]);
    c->parent = (int32_t*)(b + L.off[3]);
    c->arrive = (int32_t*)(b + L.off[4]);
    c->mom64 = (double4*)(b + L.off[5]);
    c->grp_first = (int32_t*)(b + L.off[6]);
    c->grp_n = (int32_t*)(b + L.off[7]);
    c->grp_self = (uint8_t*)(b + L.off[8]);
    c->list_off = (int64_t*)(b + L.off[9]);
    c->st_epj_off = (int64_t*)(b + L.off[10]);
    c->st_spj_off = (int64_t*)(b + L.off[11]);
    c->st_ids = (int32_t*)(b + L.off[12]);
    c->list = (int32_t*)(b + L.off[13]);
    c->items = (WorkItem*)(b + L.off[14]);
    c->order_full = (int32_t*)(b + L.off[15]);
    c->order_split = (int32_t*)(b + L.off[16]);
    c->counters = (unsigned int*)(b + L.off[17]);
    c->err = (unsigned int*)(b + L.off[18]);
    c->vel = (float4*)(b + L.off[19]);
    c->cell_lr = (int2*)(b + L.off[39]);
    c->leaf_P = (double4*)(b + L.off[40]);
    c->leaf_toff = (double4*)(b + L.off[41]);
    {
        BuildBuffers& q = c->bb;
        q.store = c->store; q.vel = c->vel; q.tmp16 = c->accp;
        q.key_a = (uint64_t*)(b + L.off[20]); q.key_b = (uint64_t*)(b + L.off[21]);
        q.idx_a = (int32_t*)(b + L.off[22]); q.idx_b = (int32_t*)(b + L.off[23]);
        q.hist = (int32_t*)(b + L.off[24]); q.scan_scratch = (int32_t*)(b + L.off[25]); q.scan_scratch64 = (int64_t*)(b + L.off[26]);
        q.bbox_part = (float*)(b + L.off[27]); q.root = (double*)(b + L.off[28]);
        q.cells = c->cells; q.geom = (double4*)(b + L.off[29]); q.parent = c->parent;
        q.level_cnt = (int32_t*)(b + L.off[30]); q.level_cap = p->max_cell + 2;
        q.mark = (int32_t*)(b + L.off[31]); q.grp_cell = (int32_t*)(b + L.off[32]);
        q.grp_first = c->grp_first; q.grp_n = c->grp_n; q.grp_box = (float*)(b + L.off[33]);
        q.n_epj = (int32_t*)(b + L.off[34]); q.n_spj = (int32_t*)(b + L.off[35]);
        q.list_off = c->list_off; q.epj_off = c->st_epj_off; q.spj_off = c->st_spj_off; q.list = c->list;
        q.walk_stacks = (int32_t*)(b + L.off[36]); q.walk_counter = (unsigned int*)(b + L.off[37]); q.err = c->err;
        q.level_bounds = (int32_t*)(b + L.off[38]);
        c->walk_warps_n = walk_warps(p->max_group);
    }
    c->max_items = max_items_of(*p);
    c->tag_groups.assign(MWF_MAX_TAG, 0);
    bool ok = true;
    // Tag t's stream gets a priority that falls with t (the device has few levels: tags share them in order), so that the
    // kernels of tags dispatched together finish roughly in tag order instead of all at the end: the retrieve of tag t (and,
    // in the pipelined loop, the upload of its next particles) then overlaps the kernels of the tags behind it.
    int prio_least = 0, prio_greatest = 0;
    ok = ok && cudaDeviceGetStreamPriorityRange(&prio_least, &prio_greatest) == cudaSuccess;
    const int prio_levels = prio_least - prio_greatest + 1;
    for (int t = 0; t < p->n_tag && ok; ++t) {
        ok = ok && cudaStreamCreateWithPriority(&c->tag_stream[t], cudaStreamNonBlocking, prio_greatest + t * prio_levels / p->n_tag) == cudaSuccess;
        c->tag_own[t] = ok;
        ok = ok && cudaEventCreateWithFlags(&c->ev_tag[t], cudaEventDisableTiming) == cudaSuccess;
        ok = ok && cudaEventCreate(&c->ev_k0[t]) == cudaSuccess;
        ok = ok && cudaEventCreate(&c->ev_k1[t]) == cudaSuccess;
        ok = ok && cudaEventCreate(&c->ev_kq[t]) == cudaSuccess;
    }
    ok = ok && cudaEventCreateWithFlags(&c->ev_store, cudaEventDisableTiming) == cudaSuccess;
    ok = ok && cudaEventCreateWithFlags(&c->ev_next, cudaEventDisableTiming) == cudaSuccess;
    ok = ok && cudaMemset(c->counters, 0, N_COUNTER * 4) == cudaSuccess;
    ok = ok && cudaMemset(c->err, 0, 256) == cudaSuccess;
    if (!ok) { mwf_destroy(c); return MWF_ECUDA; }
    *out = c;
    return MWF_OK;
}

int mwf_destroy(mwf_ctx* c) {
    if (c && c->sph) { cudaFree(c->sph); c->sph = nullptr; }
    if (!c) return MWF_EINVAL;
    cudaDeviceSynchronize();
    for (int t = 0; t < MWF_MAX_TAG; ++t) {
        if (c->tag_own[t] && c->tag_stream[t]) cudaStreamDestroy(c->tag_stream[t]);
        if (c->ev_tag[t]) cudaEventDestroy(c->ev_tag[t]);
        if (c->ev_k0[t]) cudaEventDestroy(c->ev_k0[t]);
        if (c->ev_k1[t]) cudaEventDestroy(c->ev_k1[t]);
        if (c->ev_kq[t]) cudaEventDestroy(c->ev_kq[t]);
    }
    if (c->quad64) cudaFree(c->quad64);
    if (c->quad) cudaFree(c->quad);
    if (c->ev_store) cudaEventDestroy(c->ev_store);
    if (c->ev_next) cudaEventDestroy(c->ev_next);
    for (int t = 0; t < MWF_MAX_TAG; ++t) {
        if (c->data_buf[t]) cudaFree(c->data_buf[t]);
        if (c->data_off[t]) cudaFree(c->data_off[t]);
    }
    if (c->own_arena && c->arena) cudaFree(c->arena);
    delete c;
    return MWF_OK;
}

int mwf_set_tag_stream(mwf_ctx* c, int32_t tag, void* cuda_stream) {
    if (!c || tag < 0 || tag >= c->p.n_tag) return MWF_EINVAL;
    if (c->tag_inflight[tag] || !c->tag_ranges[tag].empty()) return MWF_ESTATE;
    if (c->tag_own[tag] && c->tag_stream[tag]) cudaStreamDestroy(c->tag_stream[tag]);
    c->tag_own[tag] = false;
    c->tag_stream[tag] = static_cast<cudaStream_t>(cuda_stream);
    return MWF_OK;
}

int mwf_set_particles(mwf_ctx* c, const mwf_posm* src, int64_t first, int64_t n, int src_on_device, void* stream) {
    if (!c || !src || first < 0 || n < 0) return MWF_EINVAL;
    if (first + n > c->p.max_ptcl) return MWF_ENOMEM;
    if (c->have_tree && first + n > c->n_ptcl) return MWF_ERANGE;  // [N, ..) holds the SPJ block
    if (n == 0) return MWF_OK;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    int rc = before_store_op(c, s);
    if (rc) return rc;
    CU(c, cudaMemcpyAsync(c->store + first, src, (size_t)n * 16, src_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, s));
    c->ptcl_hi = std::max(c->ptcl_hi, first + n);
    if (c->have_tree) c->ptcl_hi = std::min(c->ptcl_hi, c->n_ptcl);
    c->mono_fresh = false;
    c->acc_full = false;
    return after_store_op(c, s);
}

int mwf_set_particles_next(mwf_ctx* c, const mwf_posm* src, int64_t first, int64_t n, int src_on_device, void* stream) {
    if (!c || !src || first < 0 || n < 0) return MWF_EINVAL;
    if (!c->have_tree) return MWF_ESTATE;
    if (first + n > c->n_ptcl) return MWF_ERANGE;
    if (n == 0) return MWF_OK;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    // no kernel reads the shadow store: its last readers were retrieved before the swap that made it the shadow
    CU(c, cudaMemcpyAsync(c->store_next + first, src, (size_t)n * 16, src_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, s));
    c->next_count += n;
    if (std::find(c->next_streams.begin(), c->next_streams.end(), s) == c->next_streams.end()) c->next_streams.push_back(s);
    return MWF_OK;
}

int mwf_swap_store(mwf_ctx* c, void* stream) {
    if (!c) return MWF_EINVAL;
    if (!c->have_tree || c->next_count != c->n_ptcl) return MWF_ESTATE;
    for (int t = 0; t < c->p.n_tag; ++t)
        if (c->tag_inflight[t] || !c->tag_ranges[t].empty()) return MWF_ESTATE;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    int rc = before_store_op(c, s);  // behind whatever still writes or reads the current store
    if (rc) return rc;
    for (cudaStream_t u : c->next_streams) {
        if (u == s) continue;
        CU(c, cudaEventRecord(c->ev_next, u));
        CU(c, cudaStreamWaitEvent(s, c->ev_next, 0));
    }
    std::swap(c->store, c->store_next);
    c->bb.store = c->store;
    c->next_count = 0;
    c->next_streams.clear();
    c->ptcl_hi = c->n_ptcl;
    c->mono_fresh = false;
    c->acc_full = false;
    return after_store_op(c, s);  // every later dispatch / store operation waits for this event, hence for the uploads
}

int mwf_get_tag_split(mwf_ctx* c, int64_t* bounds) {
    if (!c || !bounds) return MWF_EINVAL;
    if (!c->have_lists) return MWF_ESTATE;
    for (int t = 0; t <= c->p.n_tag; ++t) bounds[t] = c->h_split[(size_t)t];
    return MWF_OK;
}

int mwf_get_particles(mwf_ctx* c, mwf_posm* dst, int64_t first, int64_t n, int dst_on_device) {
    if (!c || !dst || first < 0 || n < 0 || first + n > c->p.max_ptcl) return MWF_EINVAL;
    CU(c, cudaDeviceSynchronize());
    CU(c, cudaMemcpy(dst, c->store + first, (size_t)n * 16, dst_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost));
    return MWF_OK;
}

int mwf_set_tree(mwf_ctx* c, const mwf_cell* cells, int64_t n_cell, void* stream) {
    if (!c || !cells || n_cell < 1) return MWF_EINVAL;
    if (n_cell > c->p.max_cell) return MWF_ENOMEM;
    const int64_t n = cells[0].n_ptcl;
    if (n < 1) return MWF_ERANGE;
    if (n > c->p.max_ptcl) return MWF_ENOMEM;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    int rc = before_store_op(c, s);
    if (rc) return rc;
    c->have_tree = false;
    c->built_on_device = false;
    drop_lists(c);
    c->mono_fresh = false;
    CU(c, cudaMemsetAsync(c->err, 0, sizeof(unsigned int), s));
    CU(c, cudaMemcpyAsync(c->cells, cells, (size_t)n_cell * sizeof(mwf_cell), cudaMemcpyHostToDevice, s));
    CU(c, launch_tree_prepare(c->cells, n_cell, c->p.max_ptcl, c->parent, c->arrive, c->err, s));
    ++c->n_launch;
    {   // a tree that failed the validation must not be ranked (its ranges may point anywhere)
        unsigned int e0 = 0;
        rc = read_err_word(c, s, &e0);
        if (rc) return rc;
        if (e0) { after_store_op(c, s); return MWF_ERANGE; }
    }
    CU(c, launch_leaf_ranking(c->cells, n_cell, n, c->bb.mark, c->bb.scan_scratch, c->cell_lr, &c->n_leaf_cells, s));
    c->n_launch += 5;
    // zero-mass dummy record behind the SPJ block: what list padding points at
    const float4 zero = make_float4(0.f, 0.f, 0.f, 0.f);
    CU(c, cudaMemcpyAsync(c->store + n + n_cell, &zero, 16, cudaMemcpyHostToDevice, s));
    CU(c, cudaMemcpyAsync(c->store_next + n + n_cell, &zero, 16, cudaMemcpyHostToDevice, s));
    c->next_count = 0;
    c->next_streams.clear();
    unsigned int e = 0;
    rc = read_err_word(c, s, &e);
    if (rc) return rc;
    rc = after_store_op(c, s);
    if (rc) return rc;
    if (e) return MWF_ERANGE;
    c->n_ptcl = n;
    c->n_cell = n_cell;
    c->ptcl_hi = std::min(c->ptcl_hi, n);
    c->have_tree = true;
    return MWF_OK;
}

int mwf_set_lists(mwf_ctx* c, int64_t n_group, const int32_t* grp_first, const int32_t* grp_n, const int64_t* epj_off,
                  const int32_t* epj_id, const int64_t* spj_off, const int32_t* spj_id, int mode, void* stream) {
    if (!c || n_group < 1 || !grp_first || !grp_n || !epj_off || !spj_off) return MWF_EINVAL;
    if (mode != MWF_MAKE_LIST && mode != MWF_MAKE_LIST_FOR_REUSE) return MWF_EINVAL;
    if (!c->have_tree) return MWF_ESTATE;
    if (n_group > c->p.max_group) return MWF_ENOMEM;
    if (epj_off[0] != 0 || spj_off[0] != 0) return MWF_ERANGE;
    const int64_t e_epj = epj_off[n_group], e_spj = spj_off[n_group];
    if (e_epj < 0 || e_spj < 0) return MWF_ERANGE;
    if ((e_epj > 0 && !epj_id) || (e_spj > 0 && !spj_id)) return MWF_EINVAL;
    if (e_epj + e_spj > c->p.max_entry) return MWF_ENOMEM;
    // host pass: offsets, items, schedule
    std::vector<int64_t> n_list((size_t)n_group);
    for (int64_t g = 0; g < n_group; ++g) {
        const int64_t ne = epj_off[g + 1] - epj_off[g], ns = spj_off[g + 1] - spj_off[g];
        if (ne < 0 || ns < 0) return MWF_ERANGE;
        n_list[(size_t)g] = ne + ns;
    }
    Plan plan;
    {
        const int prc = make_plan(c, n_group, grp_first, grp_n, n_list.data(), plan);
        if (prc) return prc;
    }
    const std::vector<int64_t>& list_off = plan.list_off;
    const std::vector<WorkItem>& items = plan.items;
    const std::vector<int32_t>& order_full = plan.order_full;
    const int64_t n_items = (int64_t)items.size();
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    int rc = before_store_op(c, s);
    if (rc) return rc;
    drop_lists(c);
    const auto H2D = cudaMemcpyHostToDevice;
    CU(c, cudaMemsetAsync(c->err, 0, sizeof(unsigned int), s));
    CU(c, cudaMemcpyAsync(c->grp_first, grp_first, (size_t)n_group * 4, H2D, s));
    CU(c, cudaMemcpyAsync(c->grp_n, grp_n, (size_t)n_group * 4, H2D, s));
    CU(c, cudaMemcpyAsync(c->st_epj_off, epj_off, (size_t)(n_group + 1) * 8, H2D, s));
    CU(c, cudaMemcpyAsync(c->st_spj_off, spj_off, (size_t)(n_group + 1) * 8, H2D, s));
    if (e_epj) CU(c, cudaMemcpyAsync(c->st_ids, epj_id, (size_t)e_epj * 4, H2D, s));
    if (e_spj) CU(c, cudaMemcpyAsync(c->st_ids + e_epj, spj_id, (size_t)e_spj * 4, H2D, s));
    CU(c, cudaMemcpyAsync(c->list_off, list_off.data(), (size_t)(n_group + 1) * 8, H2D, s));
    CU(c, cudaMemcpyAsync(c->items, items.data(), (size_t)n_items * sizeof(WorkItem), H2D, s));
    CU(c, cudaMemcpyAsync(c->order_full, order_full.data(), (size_t)n_items * 4, H2D, s));
    CU(c, launch_merge_lists(n_group, c->grp_first, c->grp_n, c->st_epj_off, c->st_ids, c->st_spj_off, c->st_ids + e_epj, c->list_off,
                             c->n_ptcl, c->n_cell, c->list, c->grp_self, c->err, s));
    ++c->n_launch;
    unsigned int e = 0;
    rc = read_err_word(c, s, &e);  // also makes the host vectors above safe to free
    if (rc) return rc;
    rc = after_store_op(c, s);
    if (rc) return rc;
    if (e & ~ERR_SELF_MIXED) return MWF_ERANGE;
    if (e) return MWF_EINVAL;  // only the self-membership rule is violated
    adopt_plan(c, plan, n_group, grp_first, grp_n, mode);
    return MWF_OK;
}

int mwf_begin_step(mwf_ctx* c, int mode) {
    if (!c) return MWF_EINVAL;
    if (mode == MWF_REUSE_LIST) {
        if (!c->have_lists || !c->lists_for_reuse) return MWF_ESTATE;  // MAKE_LIST keeps nothing
        c->groups_dispatched = 0;
        return MWF_OK;
    }
    if (mode == MWF_MAKE_LIST || mode == MWF_MAKE_LIST_FOR_REUSE) {
        for (int t = 0; t < c->p.n_tag; ++t)
            if (!c->tag_ranges[t].empty()) return MWF_ESTATE;  // results of the previous step not retrieved
        drop_lists(c);
        return MWF_OK;
    }
    return MWF_EINVAL;
}

int mwf_refresh_monopoles(mwf_ctx* c, void* stream) {
    if (!c) return MWF_EINVAL;
    if (!c->have_tree || c->ptcl_hi < c->n_ptcl) return MWF_ESTATE;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    int rc = before_store_op(c, s);
    if (rc) return rc;
    if (c->spj_order == 2 || !use_scan_refresh()) {  // the quadrupoles need the bottom-up pass (parallel-axis theorem)
        CU(c, launch_monopoles(c->cells, c->parent, c->n_cell, c->n_ptcl, c->store, c->mom64, c->arrive,
                               c->spj_order == 2 ? c->quad64 : nullptr, c->spj_order == 2 ? c->quad : nullptr, s));
        ++c->n_launch;
    } else {
        CU(c, launch_monopoles_scan(c->cells, c->cell_lr, c->n_cell, c->n_ptcl, c->n_leaf_cells, c->store, c->leaf_P, c->leaf_toff, s));
        c->n_launch += 4;
    }
    c->mono_fresh = true;
    return after_store_op(c, s);
}

// The schedule of a dispatch over groups [g_begin, g_end): the full one, a per-tag one, or none (item order).
static int pick_order(mwf_ctx* c, int64_t g_begin, int64_t g_end, cudaStream_t s, const int32_t** order) {
    *order = nullptr;
    if (g_begin == 0 && g_end == c->n_group) {
        *order = c->order_full;
        return MWF_OK;
    }
    for (int t = 0; t < c->p.n_tag; ++t)
        if (c->h_split[(size_t)t] == g_begin && c->h_split[(size_t)t + 1] == g_end) {
            const int rc = ensure_split_order(c, s);
            if (rc) return rc;
            *order = c->order_split;
        }
    return MWF_OK;
}

// Bookkeeping common to every kind of dispatch: the tag is in flight, its particle ranges await a retrieve.
static void book_dispatch(mwf_ctx* c, int32_t tag, int64_t g_begin, int64_t g_end) {
    c->tag_inflight[tag] = true;
    ++c->n_launch;
    c->n_inter += c->h_inter[(size_t)g_end] - c->h_inter[(size_t)g_begin];
    // particle range covered (groups are disjoint; contiguous when they come from a tree)
    int64_t lo = c->h_grp_first[(size_t)g_begin], hi = lo + c->h_grp_n[(size_t)g_begin];
    auto& rs = c->tag_ranges[tag];
    for (int64_t g = g_begin + 1; g < g_end; ++g) {
        const int64_t f = c->h_grp_first[(size_t)g], n = c->h_grp_n[(size_t)g];
        if (f == hi) { hi += n; continue; }
        rs.emplace_back(lo, hi);
        lo = f; hi = f + n;
    }
    rs.emplace_back(lo, hi);
    c->tag_groups[(size_t)tag] += g_end - g_begin;
    c->groups_outstanding += g_end - g_begin;
}

// Launch of the force kernel over groups [g_begin, g_end) on the tag's stream and the bookkeeping that goes with it.
// jdata / joff (device) non-null: method G1, the lists are runs of j records instead of indices into the store.
static int dispatch_launch(mwf_ctx* c, int32_t tag, int64_t g_begin, int64_t g_end, const float4* jdata, const int64_t* joff) {
    cudaStream_t s = c->tag_stream[tag];
    ForceArgs a;
    a.store = c->store;
    a.list = c->list;
    a.list_off = c->list_off;
    a.grp_self = c->grp_self;
    a.items = c->items;
    a.jdata = jdata;
    a.joff = joff;
    a.g_base = g_begin;
    a.accp = c->accp;
    a.item_begin = c->h_item_off[(size_t)g_begin];
    a.n_items = c->h_item_off[(size_t)g_end] - a.item_begin;
    a.eps2 = c->p.eps * c->p.eps;
    a.G = c->p.G;
    {
        const int rc = pick_order(c, g_begin, g_end, s, &a.order);
        if (rc) return rc;
    }
    const int64_t resident = (int64_t)c->n_sm * c->ctas_per_sm;
    const int64_t want = (a.n_items + WARPS_PER_CTA - 1) / WARPS_PER_CTA;
    int grid = (int)resident, warps = WARPS_PER_CTA;
    a.counter = nullptr;
    if (want > resident) {  // more items than resident warps: claim the rest dynamically
        a.counter = c->counters + (c->counter_seq++ % N_COUNTER);
        CU(c, cudaMemsetAsync(a.counter, 0, sizeof(unsigned int), s));
    } else {  // sub-wave dispatch: one item per warp, small blocks (see launch_force)
        warps = SMALL_CTA_WARPS;
        grid = (int)((a.n_items + warps - 1) / warps);
    }
    CU(c, cudaEventRecord(c->ev_k0[tag], s));
    CU(c, launch_force(a, grid, warps, s));
    c->tag_quad[tag] = false;
    if (c->spj_order == 2) {  // quadrupole terms of the SPJ entries, added behind the monopole kernel
        QuadArgs q;
        q.store = c->store; q.quad = c->quad; q.list = c->list; q.list_off = c->list_off;
        q.epj_off = c->st_epj_off; q.spj_off = c->st_spj_off;
        q.items = c->items; q.order = a.order; q.accp = c->accp;
        q.item_begin = a.item_begin; q.n_items = a.n_items; q.n_ptcl = c->n_ptcl; q.eps2 = a.eps2; q.G = a.G;
        const int64_t qres = (int64_t)c->n_sm * c->quad_ctas_per_sm;
        const int qgrid = (int)std::min(want, qres);
        q.counter = nullptr;
        if (want > qres) {
            q.counter = c->counters + (c->counter_seq++ % N_COUNTER);
            CU(c, cudaMemsetAsync(q.counter, 0, sizeof(unsigned int), s));
        }
        CU(c, cudaEventRecord(c->ev_kq[tag], s));
        CU(c, launch_quad(q, qgrid, s));
        c->tag_quad[tag] = true;
        ++c->n_launch;
    }
    CU(c, cudaEventRecord(c->ev_k1[tag], s));
    CU(c, cudaEventRecord(c->ev_tag[tag], s));
    c->tag_timed[tag] = true;
    book_dispatch(c, tag, g_begin, g_end);
    c->groups_dispatched += g_end - g_begin;
    if (c->groups_dispatched >= c->n_group) c->acc_full = true;
    return MWF_OK;
}

int mwf_dispatch(mwf_ctx* c, int32_t tag, int64_t g_begin, int64_t g_end) {
    if (!c || tag < 0 || tag >= c->p.n_tag || g_begin < 0 || g_end < g_begin) return MWF_EINVAL;
    if (!c->have_tree || !c->have_lists || !c->mono_fresh) return MWF_ESTATE;
    if (g_end > c->n_group) return MWF_ERANGE;
    if (g_end == g_begin) return MWF_OK;
    if (!c->tag_ranges[tag].empty() && c->tag_kind[tag] != 0) return MWF_ESTATE;  // SPH records await their retrieve
    c->tag_kind[tag] = 0;
    if (c->store_event_valid) CU(c, cudaStreamWaitEvent(c->tag_stream[tag], c->ev_store, 0));
    return dispatch_launch(c, tag, g_begin, g_end, nullptr, nullptr);
}

int mwf_reserve_data_lists(mwf_ctx* c, int64_t max_entry_per_tag) {
    if (!c || max_entry_per_tag < 1) return MWF_EINVAL;
    for (int t = 0; t < c->p.n_tag; ++t)
        if (c->tag_inflight[t] || !c->tag_ranges[t].empty()) return MWF_ESTATE;
    CU(c, cudaDeviceSynchronize());
    for (int t = 0; t < c->p.n_tag; ++t) {
        if (c->data_buf[t]) { cudaFree(c->data_buf[t]); c->data_buf[t] = nullptr; }
        if (c->data_off[t]) { cudaFree(c->data_off[t]); c->data_off[t] = nullptr; }
    }
    c->data_cap = 0;
    for (int t = 0; t < c->p.n_tag; ++t) {
        void *a = nullptr, *b = nullptr;
        if (cudaMalloc(&a, (size_t)max_entry_per_tag * 16) != cudaSuccess || cudaMalloc(&b, (size_t)(c->p.max_group + 1) * 8) != cudaSuccess) {
            cudaGetLastError();
            if (a) cudaFree(a);
            return MWF_ENOMEM;
        }
        c->data_buf[t] = static_cast<float4*>(a);
        c->data_off[t] = static_cast<int64_t*>(b);
    }
    c->data_cap = max_entry_per_tag;
    return MWF_OK;
}

int mwf_dispatch_data(mwf_ctx* c, int32_t tag, int64_t g_begin, int64_t g_end, const mwf_posm* jdata, const int64_t* joff, int jdata_on_device) {
    if (!c || tag < 0 || tag >= c->p.n_tag || g_begin < 0 || g_end < g_begin || !jdata || !joff) return MWF_EINVAL;
    if (!c->have_tree || !c->have_lists || c->data_cap < 1 || c->spj_order != 1) return MWF_ESTATE;
    if (c->ptcl_hi < c->n_ptcl) return MWF_ESTATE;  // the i-particles are read from the store
    if (g_end > c->n_group) return MWF_ERANGE;
    if (g_end == g_begin) return MWF_OK;
    if (c->tag_inflight[tag]) return MWF_ESTATE;  // the tag's staging buffer is still being read: retrieve first
    c->tag_kind[tag] = 0;
    const int64_t ng = g_end - g_begin;
    if (joff[0] != 0) return MWF_ERANGE;
    for (int64_t g = 0; g < ng; ++g)  // the run of group g_begin + g must be as long as the group's index list
        if (joff[g + 1] - joff[g] != (c->h_inter[(size_t)(g_begin + g) + 1] - c->h_inter[(size_t)(g_begin + g)]) / c->h_grp_n[(size_t)(g_begin + g)])
            return MWF_ERANGE;
    if (joff[ng] > c->data_cap) return MWF_ENOMEM;
    cudaStream_t s = c->tag_stream[tag];
    if (c->store_event_valid) CU(c, cudaStreamWaitEvent(s, c->ev_store, 0));
    CU(c, cudaMemcpyAsync(c->data_off[tag], joff, (size_t)(ng + 1) * 8, cudaMemcpyHostToDevice, s));
    if (joff[ng] > 0)
        CU(c, cudaMemcpyAsync(c->data_buf[tag], jdata, (size_t)joff[ng] * 16, jdata_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, s));
    return dispatch_launch(c, tag, g_begin, g_end, c->data_buf[tag], c->data_off[tag]);
}

int mwf_retrieve(mwf_ctx* c, int32_t tag, mwf_accp* dst, int dst_on_device) {
    if (!c || tag < 0 || tag >= c->p.n_tag) return MWF_EINVAL;
    auto& rs = c->tag_ranges[tag];
    if (rs.empty()) return MWF_ESTATE;
    cudaStream_t s = c->tag_stream[tag];
    const auto kind = dst_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
    // merge adjacent ranges of consecutive dispatches
    std::sort(rs.begin(), rs.end());
    size_t k = dst ? 0 : rs.size();  // dst == NULL: wait for the tag and discard its results
    while (k < rs.size()) {
        int64_t lo = rs[k].first, hi = rs[k].second;
        size_t j = k + 1;
        while (j < rs.size() && rs[j].first <= hi) { hi = std::max(hi, rs[j].second); ++j; }
        const float4* from = c->tag_kind[tag] == 1 ? c->sph : c->accp;
        CU(c, cudaMemcpyAsync(reinterpret_cast<float4*>(dst) + lo, from + lo, (size_t)(hi - lo) * 16, kind, s));
        k = j;
    }
    CU(c, cudaStreamSynchronize(s));
    rs.clear();
    c->tag_inflight[tag] = false;
    c->groups_outstanding -= c->tag_groups[(size_t)tag];
    c->tag_groups[(size_t)tag] = 0;
    // MAKE_LIST: the lists served their one evaluation
    if (c->have_lists && !c->lists_for_reuse && c->groups_outstanding == 0 && c->groups_dispatched >= c->n_group) drop_lists(c);
    return MWF_OK;
}

int mwf_calc_force_all(mwf_ctx* c, const mwf_posm* src, int src_on_device, mwf_accp* dst, int dst_on_device) {
    if (!c || !dst) return MWF_EINVAL;
    if (!c->have_tree || !c->have_lists) return MWF_ESTATE;
    cudaStream_t s0 = c->tag_stream[0];
    int rc;
    if (src) {
        rc = mwf_set_particles(c, src, 0, c->n_ptcl, src_on_device, s0);
        if (rc) return rc;
    }
    if (!c->mono_fresh) {
        rc = mwf_refresh_monopoles(c, s0);
        if (rc) return rc;
    }
    // host destination: one dispatch per tag so that each D2H copy overlaps the other tags' kernels
    const int n_part = dst_on_device ? 1 : c->p.n_tag;
    if (n_part == 1) {
        rc = mwf_dispatch(c, 0, 0, c->n_group);
        if (rc) return rc;
        return mwf_retrieve(c, 0, dst, dst_on_device);
    }
    bool used[MWF_MAX_TAG] = {false};
    for (int t = 0; t < n_part; ++t) {
        const int64_t gb = c->h_split[(size_t)t], ge = c->h_split[(size_t)t + 1];
        if (ge == gb) continue;
        rc = mwf_dispatch(c, t, gb, ge);
        if (rc) return rc;
        used[t] = true;
    }
    for (int t = 0; t < n_part; ++t) {
        if (!used[t]) continue;
        rc = mwf_retrieve(c, t, dst, dst_on_device);
        if (rc) return rc;
    }
    return MWF_OK;
}

// The device-side construction step behind mwf_build (opening angle theta) and mwf_build_neighbours (search radii 2 (1 + skin) h).
static int build_impl(mwf_ctx* c, int64_t n, int32_t n_leaf, int32_t n_grp, double theta, bool neighbours, double skin, int mode, void* stream) {
    if (!c || n < 1 || n_leaf < 1 || n_grp < 1) return MWF_EINVAL;
    if (neighbours ? !(skin >= 0.0) : (!(theta >= 0.0) || theta > 1.0)) return MWF_EINVAL;
    if (mode != MWF_MAKE_LIST && mode != MWF_MAKE_LIST_FOR_REUSE) return MWF_EINVAL;
    if (n > c->p.max_ptcl) return MWF_ENOMEM;
    if (neighbours && (!c->sph || c->sph_hi < n)) return MWF_ESTATE;  // the smoothing lengths of particles [0, n) must have been uploaded
    if (c->ptcl_hi < n && !(c->have_tree && c->n_ptcl >= n)) return MWF_ESTATE;  // particles [0, n) must have been uploaded
    for (int t = 0; t < c->p.n_tag; ++t)
        if (!c->tag_ranges[t].empty()) return MWF_ESTATE;  // tmp16 aliases the result array: retrieve first
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    int rc = before_store_op(c, s);
    if (rc) return rc;
    c->have_tree = false;
    c->built_on_device = false;
    drop_lists(c);
    c->mono_fresh = false;
    CU(c, cudaMemsetAsync(c->err, 0, sizeof(unsigned int), s));
    const bool with_vel = c->vel_hi >= n;
    int64_t n_cell = 0, n_group = 0;
    int n_level = 0;
    PhaseTimer tm;
    float4* sph = (c->sph && c->sph_hi >= n) ? c->sph : nullptr;
    CU(c, build_tree_device(c->bb, n, n_leaf, n_grp, c->p.max_cell, c->p.max_group, with_vel, sph, &n_cell, &n_group, &n_level, s));
    c->n_launch += 8 + 3 * 8 + 3 * n_level;
    tm.lap("sort + tree + groups");
    if (n_cell > c->p.max_cell || n_group > c->p.max_group) { after_store_op(c, s); return MWF_ENOMEM; }
    unsigned int e = 0;
    rc = read_err_word(c, s, &e);
    if (rc) return rc;
    if (e) { after_store_op(c, s); return MWF_ENOMEM; }
    // tree state as mwf_set_tree leaves it: arrival counters zero, leaves ranked, dummy record behind the SPJ block
    CU(c, cudaMemsetAsync(c->arrive, 0, (size_t)n_cell * 4, s));
    CU(c, launch_leaf_ranking(c->cells, n_cell, n, c->bb.mark, c->bb.scan_scratch, c->cell_lr, &c->n_leaf_cells, s));
    c->n_launch += 5;
    const float4 zero = make_float4(0.f, 0.f, 0.f, 0.f);
    CU(c, cudaMemcpyAsync(c->store + n + n_cell, &zero, 16, cudaMemcpyHostToDevice, s));
    CU(c, cudaMemcpyAsync(c->store_next + n + n_cell, &zero, 16, cudaMemcpyHostToDevice, s));
    c->next_count = 0;
    c->next_streams.clear();
    c->n_ptcl = n;
    c->n_cell = n_cell;
    c->ptcl_hi = n;
    // lists: counting walk, offsets, capacity check, fill walk
    int64_t padded = 0, e_epj = 0, e_spj = 0;
    WalkRule rule;
    rule.theta = theta;
    if (neighbours) {  // per-cell and per-group search radii; level_cnt and mark are free once the tree and the groups exist
        rule.neighbours = true;
        rule.reach = 2.0 * (1.0 + skin);
        rule.cell_h = reinterpret_cast<float*>(c->bb.level_cnt);
        rule.grp_h = reinterpret_cast<float*>(c->bb.mark);
        CU(c, build_smoothing_reach(c->bb, c->sph, n_cell, n_group, reinterpret_cast<float*>(c->bb.level_cnt), reinterpret_cast<float*>(c->bb.mark), s));
        c->n_launch += 2;
    }
    CU(c, build_lists_count(c->bb, n_group, rule, c->walk_warps_n, &padded, &e_epj, &e_spj, s));
    tm.lap("list walk: count + offsets");
    if (e_epj + e_spj > c->p.max_entry) { after_store_op(c, s); return MWF_ENOMEM; }
    // group sizes and list lengths come back for the host work plan; the fill walk runs meanwhile
    std::vector<int32_t> h_first((size_t)n_group), h_n((size_t)n_group), h_ne((size_t)n_group), h_ns((size_t)n_group);
    const auto D2H = cudaMemcpyDeviceToHost;
    CU(c, cudaMemcpyAsync(h_first.data(), c->grp_first, (size_t)n_group * 4, D2H, s));
    CU(c, cudaMemcpyAsync(h_n.data(), c->grp_n, (size_t)n_group * 4, D2H, s));
    CU(c, cudaMemcpyAsync(h_ne.data(), c->bb.n_epj, (size_t)n_group * 4, D2H, s));
    CU(c, cudaMemcpyAsync(h_ns.data(), c->bb.n_spj, (size_t)n_group * 4, D2H, s));
    CU(c, cudaStreamSynchronize(s));
    CU(c, build_lists_fill(c->bb, n_group, rule, c->walk_warps_n, n, n_cell, s));
    CU(c, cudaMemsetAsync(c->grp_self, 1, (size_t)n_group, s));  // theta <= 1: a group's own cells are always opened
    c->n_launch += 6;
    std::vector<int64_t> n_list((size_t)n_group);
    for (int64_t g = 0; g < n_group; ++g) n_list[(size_t)g] = (int64_t)h_ne[(size_t)g] + h_ns[(size_t)g];
    Plan plan;
    rc = make_plan(c, n_group, h_first.data(), h_n.data(), n_list.data(), plan);
    tm.lap("host work plan | fill walk");
    if (rc) { after_store_op(c, s); return rc; }
    if (plan.list_off[(size_t)n_group] != padded) { after_store_op(c, s); return MWF_ERANGE; }  // host and device offsets must agree
    const int64_t n_items = (int64_t)plan.items.size();
    const auto H2D = cudaMemcpyHostToDevice;
    CU(c, cudaMemcpyAsync(c->items, plan.items.data(), (size_t)n_items * sizeof(WorkItem), H2D, s));
    CU(c, cudaMemcpyAsync(c->order_full, plan.order_full.data(), (size_t)n_items * 4, H2D, s));
    CU(c, cudaStreamSynchronize(s));  // the plan's host vectors die with this call
    tm.lap("plan upload");
    rc = after_store_op(c, s);
    if (rc) return rc;
    c->have_tree = true;
    c->built_on_device = true;
    c->build_e_epj = e_epj;
    c->build_e_spj = e_spj;
    c->build_n_level = n_level;
    adopt_plan(c, plan, n_group, h_first.data(), h_n.data(), mode);
    return MWF_OK;
}

int mwf_build(mwf_ctx* c, int64_t n, int32_t n_leaf, int32_t n_grp, double theta, int mode, void* stream) {
    return build_impl(c, n, n_leaf, n_grp, theta, false, 0.0, mode, stream);
}

int mwf_build_neighbours(mwf_ctx* c, int64_t n, int32_t n_leaf, int32_t n_grp, double skin, int mode, void* stream) {
    return build_impl(c, n, n_leaf, n_grp, 0.0, true, skin, mode, stream);
}

int mwf_get_build_sizes(mwf_ctx* c, int64_t* n_cell, int64_t* n_group, int64_t* n_epj, int64_t* n_spj, int32_t* n_level) {
    if (!c) return MWF_EINVAL;
    if (!c->built_on_device || !c->have_lists) return MWF_ESTATE;
    if (n_cell) *n_cell = c->n_cell;
    if (n_group) *n_group = c->n_group;
    if (n_epj) *n_epj = c->build_e_epj;
    if (n_spj) *n_spj = c->build_e_spj;
    if (n_level) *n_level = c->build_n_level;
    return MWF_OK;
}

int mwf_get_permutation(mwf_ctx* c, int32_t* perm, int dst_on_device) {
    if (!c || !perm) return MWF_EINVAL;
    if (!c->built_on_device) return MWF_ESTATE;
    CU(c, cudaDeviceSynchronize());
    CU(c, cudaMemcpy(perm, c->bb.idx_a, (size_t)c->n_ptcl * 4, dst_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost));
    return MWF_OK;
}

int mwf_get_tree(mwf_ctx* c, mwf_cell* cells, double* geom4) {
    if (!c || (!cells && !geom4)) return MWF_EINVAL;
    if (!c->have_tree) return MWF_ESTATE;
    if (geom4 && !c->built_on_device) return MWF_ESTATE;  // an uploaded tree carries no geometry
    CU(c, cudaDeviceSynchronize());
    if (cells) CU(c, cudaMemcpy(cells, c->cells, (size_t)c->n_cell * sizeof(mwf_cell), cudaMemcpyDeviceToHost));
    if (geom4) CU(c, cudaMemcpy(geom4, c->bb.geom, (size_t)c->n_cell * 32, cudaMemcpyDeviceToHost));
    return MWF_OK;
}

int mwf_get_groups(mwf_ctx* c, int32_t* grp_first, int32_t* grp_n) {
    if (!c || !grp_first || !grp_n) return MWF_EINVAL;
    if (!c->have_lists) return MWF_ESTATE;
    std::memcpy(grp_first, c->h_grp_first.data(), (size_t)c->n_group * 4);
    std::memcpy(grp_n, c->h_grp_n.data(), (size_t)c->n_group * 4);
    return MWF_OK;
}

int mwf_get_lists(mwf_ctx* c, int64_t* epj_off, int32_t* epj_id, int64_t* spj_off, int32_t* spj_id) {
    if (!c || !epj_off || !spj_off || !epj_id || !spj_id) return MWF_EINVAL;
    if (!c->built_on_device || !c->have_lists) return MWF_ESTATE;
    CU(c, cudaDeviceSynchronize());
    // un-merge into the staging area of the upload path, then two bulk copies
    if (c->build_e_epj + c->build_e_spj > c->p.max_entry) return MWF_ENOMEM;
    int32_t* d_epj = c->st_ids;
    int32_t* d_spj = c->st_ids + c->build_e_epj;
    CU(c, unmerge_lists(c->bb, c->n_group, c->n_ptcl, d_epj, d_spj, nullptr));
    CU(c, cudaDeviceSynchronize());
    CU(c, cudaMemcpy(epj_off, c->bb.epj_off, (size_t)(c->n_group + 1) * 8, cudaMemcpyDeviceToHost));
    CU(c, cudaMemcpy(spj_off, c->bb.spj_off, (size_t)(c->n_group + 1) * 8, cudaMemcpyDeviceToHost));
    if (c->build_e_epj) CU(c, cudaMemcpy(epj_id, d_epj, (size_t)c->build_e_epj * 4, cudaMemcpyDeviceToHost));
    if (c->build_e_spj) CU(c, cudaMemcpy(spj_id, d_spj, (size_t)c->build_e_spj * 4, cudaMemcpyDeviceToHost));
    return MWF_OK;
}

int mwf_set_velocities(mwf_ctx* c, const mwf_vel* src, int64_t first, int64_t n, int src_on_device, void* stream) {
    if (!c || !src || first < 0 || n < 0) return MWF_EINVAL;
    if (first + n > c->p.max_ptcl) return MWF_ENOMEM;
    if (n == 0) return MWF_OK;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    int rc = before_store_op(c, s);
    if (rc) return rc;
    CU(c, cudaMemcpyAsync(c->vel + first, src, (size_t)n * 16, src_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, s));
    if (first <= c->vel_hi) c->vel_hi = std::max(c->vel_hi, first + n);
    return after_store_op(c, s);
}

int mwf_get_velocities(mwf_ctx* c, mwf_vel* dst, int64_t first, int64_t n, int dst_on_device) {
    if (!c || !dst || first < 0 || n < 0 || first + n > c->p.max_ptcl) return MWF_EINVAL;
    CU(c, cudaDeviceSynchronize());
    CU(c, cudaMemcpy(dst, c->vel + first, (size_t)n * 16, dst_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost));
    return MWF_OK;
}

static int integrate_ready(mwf_ctx* c, float dt) {
    if (!c || !(dt == dt)) return MWF_EINVAL;
    if (!c->have_tree || !c->have_lists || !c->acc_full || c->vel_hi < c->n_ptcl) return MWF_ESTATE;
    return MWF_OK;
}

int mwf_kick_drift(mwf_ctx* c, float dt, void* stream) {
    int rc = integrate_ready(c, dt);
    if (rc) return rc;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    rc = before_store_op(c, s);  // waits for the force kernels that read the store and write accp
    if (rc) return rc;
    CU(c, launch_kick_drift(c->store, c->vel, c->accp, c->n_ptcl, dt, s));
    ++c->n_launch;
    c->mono_fresh = false;
    c->acc_full = false;
    return after_store_op(c, s);
}

int mwf_kick(mwf_ctx* c, float dt, void* stream) {
    int rc = integrate_ready(c, dt);
    if (rc) return rc;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    rc = before_store_op(c, s);
    if (rc) return rc;
    CU(c, launch_kick(c->vel, c->accp, c->n_ptcl, dt, s));
    ++c->n_launch;
    return after_store_op(c, s);
}

int mwf_step_reuse(mwf_ctx* c, float dt) {
    int rc = integrate_ready(c, dt);
    if (rc) return rc;
    for (int t = 1; t < c->p.n_tag; ++t)
        if (!c->tag_ranges[t].empty()) return MWF_ESTATE;  // results of another tag not retrieved
    rc = mwf_begin_step(c, MWF_REUSE_LIST);
    if (rc) return rc;
    cudaStream_t s0 = c->tag_stream[0];
    rc = mwf_kick_drift(c, dt, s0);
    if (rc) return rc;
    rc = mwf_refresh_monopoles(c, s0);
    if (rc) return rc;
    // results stay on the device: forget what earlier steps left for tag 0, a later retrieve copies all N
    c->groups_outstanding -= c->tag_groups[0];
    c->tag_groups[0] = 0;
    c->tag_ranges[0].clear();
    rc = mwf_dispatch(c, 0, 0, c->n_group);
    if (rc) return rc;
    return mwf_kick(c, dt, s0);
}

// ---- short-range workload (NEXT-4)

int mwf_set_sph(mwf_ctx* c, const mwf_sph* src, int64_t first, int64_t n, int src_on_device, void* stream) {
    if (!c || !src || first < 0 || n < 0) return MWF_EINVAL;
    if (first + n > c->p.max_ptcl) return MWF_ENOMEM;
    if (!c->sph) {
        void* q = nullptr;
        if (cudaMalloc(&q, (size_t)c->p.max_ptcl * 16) != cudaSuccess) { cudaGetLastError(); return MWF_ENOMEM; }
        c->sph = static_cast<float4*>(q);
        c->sph_ctas_per_sm[0] = sph_max_ctas_per_sm(false);
        c->sph_ctas_per_sm[1] = sph_max_ctas_per_sm(true);
        if (c->sph_ctas_per_sm[0] < 1 || c->sph_ctas_per_sm[1] < 1) return cuda_fail(c, cudaErrorLaunchFailure, "occupancy of the SPH kernels");
    }
    if (n == 0) return MWF_OK;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    int rc = before_store_op(c, s);
    if (rc) return rc;
    CU(c, cudaMemcpyAsync(c->sph + first, src, (size_t)n * 16, src_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, s));
    if (first <= c->sph_hi) c->sph_hi = std::max(c->sph_hi, first + n);
    return after_store_op(c, s);
}

int mwf_get_sph(mwf_ctx* c, mwf_sph* dst, int64_t first, int64_t n, int dst_on_device) {
    if (!c || !dst || first < 0 || n < 0) return MWF_EINVAL;
    if (!c->sph || first + n > c->sph_hi) return MWF_ESTATE;
    CU(c, cudaDeviceSynchronize());
    CU(c, cudaMemcpy(dst, c->sph + first, (size_t)n * 16, dst_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost));
    return MWF_OK;
}

static int sph_dispatch(mwf_ctx* c, int32_t tag, int64_t g_begin, int64_t g_end, bool hydro, float gamma) {
    if (!c || tag < 0 || tag >= c->p.n_tag || g_begin < 0 || g_end < g_begin) return MWF_EINVAL;
    if (!hydro && !(gamma > 1.f)) return MWF_EINVAL;
    if (!c->have_tree || !c->have_lists || !c->sph || c->sph_hi < c->n_ptcl || c->ptcl_hi < c->n_ptcl) return MWF_ESTATE;
    if (g_end > c->n_group) return MWF_ERANGE;
    if (g_end == g_begin) return MWF_OK;
    const int kind = hydro ? 0 : 1;
    if (!c->tag_ranges[tag].empty() && c->tag_kind[tag] != kind) return MWF_ESTATE;
    c->tag_kind[tag] = kind;
    cudaStream_t s = c->tag_stream[tag];
    if (c->store_event_valid) CU(c, cudaStreamWaitEvent(s, c->ev_store, 0));
    // the hydro kernel reads the densities of every particle in its lists: wait for the density kernels of all tags;
    // the density kernel overwrites records the hydro kernels of other tags may still be reading
    for (int t = 0; t < c->p.n_tag; ++t)
        if (t != tag && c->tag_inflight[t]) CU(c, cudaStreamWaitEvent(s, c->ev_tag[t], 0));
    SphArgs a;
    a.store = c->store; a.sph = c->sph; a.list = c->list; a.list_off = c->list_off; a.items = c->items;
    a.accp = c->accp; a.n_ptcl = c->n_ptcl; a.gamma_m1 = gamma - 1.f;
    a.item_begin = c->h_item_off[(size_t)g_begin];
    a.n_items = c->h_item_off[(size_t)g_end] - a.item_begin;
    int rc = pick_order(c, g_begin, g_end, s, &a.order);
    if (rc) return rc;
    const int64_t resident = (int64_t)c->n_sm * c->sph_ctas_per_sm[hydro ? 1 : 0];
    const int64_t want = (a.n_items + WARPS_PER_CTA - 1) / WARPS_PER_CTA;
    const int grid = (int)std::min(want, resident);
    a.counter = nullptr;
    if (want > resident) {
        a.counter = c->counters + (c->counter_seq++ % N_COUNTER);
        CU(c, cudaMemsetAsync(a.counter, 0, sizeof(unsigned int), s));
    }
    CU(c, cudaEventRecord(c->ev_k0[tag], s));
    CU(c, launch_sph(a, hydro, grid, s));
    CU(c, cudaEventRecord(c->ev_k1[tag], s));
    CU(c, cudaEventRecord(c->ev_tag[tag], s));
    c->tag_timed[tag] = true;
    c->tag_quad[tag] = false;
    book_dispatch(c, tag, g_begin, g_end);
    return MWF_OK;
}

int mwf_dispatch_density(mwf_ctx* c, int32_t tag, int64_t g_begin, int64_t g_end, float gamma) {
    return sph_dispatch(c, tag, g_begin, g_end, false, gamma);
}

int mwf_dispatch_hydro(mwf_ctx* c, int32_t tag, int64_t g_begin, int64_t g_end) {
    return sph_dispatch(c, tag, g_begin, g_end, true, 0.f);
}

int mwf_calc_sph_all(mwf_ctx* c, const mwf_posm* src, int src_on_device, mwf_sph* rec, int rec_on_device, mwf_accp* dst, int dst_on_device, float gamma) {
    if (!c || !rec || !dst) return MWF_EINVAL;
    if (!c->have_tree || !c->have_lists) return MWF_ESTATE;
    cudaStream_t s0 = c->tag_stream[0];
    int rc;
    if (src) {
        rc = mwf_set_particles(c, src, 0, c->n_ptcl, src_on_device, s0);
        if (rc) return rc;
    }
    rc = mwf_set_sph(c, rec, 0, c->n_ptcl, rec_on_device, s0);
    if (rc) return rc;
    // host destinations: one dispatch per tag so that each tag's copy overlaps the other tags' kernels
    const int n_part = (rec_on_device && dst_on_device) ? 1 : c->p.n_tag;
    for (int pass = 0; pass < 2; ++pass) {
        bool used[MWF_MAX_TAG] = {false};
        for (int t = 0; t < n_part; ++t) {
            const int64_t gb = n_part == 1 ? 0 : c->h_split[(size_t)t], ge = n_part == 1 ? c->n_group : c->h_split[(size_t)t + 1];
            if (ge == gb) continue;
            rc = pass == 0 ? mwf_dispatch_density(c, t, gb, ge, gamma) : mwf_dispatch_hydro(c, t, gb, ge);
            if (rc) return rc;
            used[t] = true;
        }
        for (int t = 0; t < n_part; ++t) {
            if (!used[t]) continue;
            rc = pass == 0 ? mwf_retrieve(c, t, reinterpret_cast<mwf_accp*>(rec), rec_on_device) : mwf_retrieve(c, t, dst, dst_on_device);
            if (rc) return rc;
        }
    }
    return MWF_OK;
}

int mwf_set_spj_order(mwf_ctx* c, int order) {
    if (!c || (order != 1 && order != 2)) return MWF_EINVAL;
    for (int t = 0; t < c->p.n_tag; ++t)
        if (c->tag_inflight[t] || !c->tag_ranges[t].empty()) return MWF_ESTATE;
    if (order == 2 && !c->quad) {
        void *a = nullptr, *b = nullptr;
        if (cudaMalloc(&a, (size_t)c->p.max_cell * 48) != cudaSuccess || cudaMalloc(&b, (size_t)c->p.max_cell * 32) != cudaSuccess) {
            cudaGetLastError();
            if (a) cudaFree(a);
            return MWF_ENOMEM;
        }
        c->quad64 = static_cast<double*>(a);
        c->quad = static_cast<float4*>(b);
        c->quad_ctas_per_sm = quad_max_ctas_per_sm();
        if (c->quad_ctas_per_sm < 1) return MWF_ECUDA;
    }
    if (order != c->spj_order) {
        c->mono_fresh = false;  // the moments on the device are those of the other order
        c->acc_full = false;
    }
    c->spj_order = order;
    return MWF_OK;
}

int mwf_get_quadrupoles(mwf_ctx* c, float* dst, int dst_on_device) {
    if (!c || !dst) return MWF_EINVAL;
    if (!c->have_tree || !c->mono_fresh || c->spj_order != 2) return MWF_ESTATE;
    CU(c, cudaDeviceSynchronize());
    CU(c, cudaMemcpy(dst, c->quad, (size_t)c->n_cell * 32, dst_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost));
    return MWF_OK;
}

int mwf_last_quad_ms(mwf_ctx* c, int32_t tag, float* ms) {
    if (!c || tag < 0 || tag >= c->p.n_tag || !ms) return MWF_EINVAL;
    if (!c->tag_timed[tag] || !c->tag_quad[tag]) return MWF_ESTATE;
    CU(c, cudaEventSynchronize(c->ev_k1[tag]));
    CU(c, cudaEventElapsedTime(ms, c->ev_kq[tag], c->ev_k1[tag]));
    return MWF_OK;
}

int mwf_get_monopoles(mwf_ctx* c, mwf_posm* dst, int dst_on_device) {
    if (!c || !dst) return MWF_EINVAL;
    if (!c->have_tree || !c->mono_fresh) return MWF_ESTATE;
    CU(c, cudaDeviceSynchronize());
    CU(c, cudaMemcpy(dst, c->store + c->n_ptcl, (size_t)c->n_cell * 16, dst_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost));
    return MWF_OK;
}

int mwf_device_pointers(mwf_ctx* c, mwf_posm** store, mwf_accp** accp) {
    if (!c) return MWF_EINVAL;
    if (store) *store = reinterpret_cast<mwf_posm*>(c->store);
    if (accp) *accp = reinterpret_cast<mwf_accp*>(c->accp);
    return MWF_OK;
}

int mwf_sync(mwf_ctx* c) {
    if (!c) return MWF_EINVAL;
    CU(c, cudaDeviceSynchronize());
    return MWF_OK;
}

int mwf_get_counters(mwf_ctx* c, int64_t* kernel_launches, int64_t* interactions, int64_t* padded_entries) {
    if (!c) return MWF_EINVAL;
    if (kernel_launches) *kernel_launches = c->n_launch;
    if (interactions) *interactions = c->n_inter;
    if (padded_entries) *padded_entries = c->padded_entries;
    return MWF_OK;
}

int mwf_last_dispatch_ms(mwf_ctx* c, int32_t tag, float* ms) {
    if (!c || tag < 0 || tag >= c->p.n_tag || !ms) return MWF_EINVAL;
    if (!c->tag_timed[tag]) return MWF_ESTATE;
    CU(c, cudaEventSynchronize(c->ev_k1[tag]));
    CU(c, cudaEventElapsedTime(ms, c->ev_k0[tag], c->ev_k1[tag]));
    return MWF_OK;
}

}  // extern "C"
