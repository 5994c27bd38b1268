// Host side of the work plan: cutting groups into warp-sized work items, list offsets, interaction counts (DESIGN.md
// section 6.1).  The order in which the items are worked on is made on the device (sched_kernel.cu).
#include <climits>
#include <numeric>

#include <algorithm>

#include "mwf_ctx.h"

#ifndef MWF_TAPER
#define MWF_TAPER 1
#endif

namespace mwf {

// How a remainder of rem < 64 particles is cut: the widths of its pieces, widest first (0-terminated).  The remainder is
// padded to a multiple of a quantum q and cut into power-of-two pieces; q is the quantum whose modelled cost is lowest (a
// coarser quantum wastes lanes, a finer one re-stages the list for one more narrow item).  A table: the rule only depends
// on rem.
struct RemainderCut { int8_t width[6]; };
static const RemainderCut* remainder_table() {
    static RemainderCut table[CHUNK_I];
    static const bool made = [] {
        for (int64_t rem = 0; rem < CHUNK_I; ++rem) {
            RemainderCut& rc = table[rem];
            for (int8_t& w : rc.width) w = 0;
            if (rem == 0) continue;
            int64_t best_q = CHUNK_I, best_cost = INT64_MAX;
            for (int64_t q = 2 * MIN_WIDTH; q <= CHUNK_I; q *= 2) {
                const int64_t padded = (rem + q - 1) / q * q;
                int64_t cst = 0;
                for (int64_t piece = CHUNK_I; piece >= 2 * MIN_WIDTH; piece /= 2)
                    if (padded & piece) cst += item_cost_per_tile((int)(piece / 2));
                if (cst < best_cost) { best_cost = cst; best_q = q; }
            }
            const int64_t padded = (rem + best_q - 1) / best_q * best_q;
            int k = 0;
            for (int64_t piece = CHUNK_I; piece >= 2 * MIN_WIDTH; piece /= 2)
                if (padded & piece) rc.width[k++] = (int8_t)(piece / 2);
        }
        return true;
    }();
    (void)made;
    return table;
}

// First half of the plan: cutting every group into work items.  Needs the group ranges only, so a device-side construction
// step runs it while its counting walk is still under way.
int plan_cut(mwf_ctx* c, int64_t n_group, const int32_t* grp_first, const int32_t* grp_n, Plan& pl) {
    pl.item_off.assign((size_t)n_group + 1, 0);
    std::vector<WorkItem>& items = pl.items;
    items.clear();
    items.reserve((size_t)(c->n_ptcl / CHUNK_I + 3 * n_group));
    const RemainderCut* cut = remainder_table();
    for (int64_t g = 0; g < n_group; ++g) {
        const int64_t gf = grp_first[g], gn = grp_n[g];
        if (gf < 0 || gn < 1 || gf + gn > c->n_ptcl) return MWF_ERANGE;
        int64_t done = 0;
        auto emit = [&](int64_t n_i, int width) {
            WorkItem it;
            it.i_first = (int32_t)(gf + done);
            it.n_i = (int32_t)n_i;
            it.group = (int32_t)g;
            it.width = width;
            done += n_i;
            items.push_back(it);
        };
        for (int64_t k = 0; k < gn / CHUNK_I; ++k) emit(CHUNK_I, CHUNK_I / 2);
        const RemainderCut& rc = cut[gn % CHUNK_I];
        for (int k = 0; rc.width[k]; ++k) emit(std::min<int64_t>(2 * rc.width[k], gn - done), rc.width[k]);
        pl.item_off[(size_t)g + 1] = (int64_t)items.size();
    }
    if ((int64_t)items.size() > c->max_items) return MWF_ENOMEM;
    return MWF_OK;
}

// The items by width class, group order inside a class (a stable counting sort), and the per-group prefix counts: made
// the first time a dispatch covers a group range that has no sorted schedule of its own (1 ms of host time for 1.4e5 items,
// which a device-side construction step followed by whole-workload dispatches never needs).
int ensure_class_order(mwf_ctx* c, cudaStream_t s) {
    if (c->cls_ready) return MWF_OK;
    const std::vector<WorkItem>& items = c->h_items;
    const int64_t n_group = c->n_group;
    for (int k = 0; k < N_WIDTH_CLASS; ++k) c->h_cls_off[k].assign((size_t)n_group + 1, 0);
    for (const WorkItem& it : items) ++c->h_cls_off[width_class(it.width)][(size_t)it.group + 1];
    c->h_cls_base[0] = 0;
    for (int k = 0; k < N_WIDTH_CLASS; ++k) {
        for (int64_t g = 0; g < n_group; ++g) c->h_cls_off[k][(size_t)g + 1] += c->h_cls_off[k][(size_t)g];
        c->h_cls_base[k + 1] = c->h_cls_base[k] + c->h_cls_off[k][(size_t)n_group];
    }
    int64_t fill[N_WIDTH_CLASS];
    for (int k = 0; k < N_WIDTH_CLASS; ++k) fill[k] = c->h_cls_base[k];
    for (size_t i = 0; i < items.size(); ++i) c->h_order_cls[fill[width_class(items[i].width)]++] = (int32_t)i;
    CU(c, cudaMemcpyAsync(c->order_cls, c->h_order_cls, items.size() * sizeof(int32_t), cudaMemcpyHostToDevice, s));
    CU(c, cudaStreamSynchronize(s));  // the other tags' streams read it too
    c->cls_ready = true;
    return MWF_OK;
}

// Second half: list offsets, interaction counts, the items' modelled costs, the schedules.  Needs the list lengths.
int plan_finish(mwf_ctx* c, int64_t n_group, const int32_t* grp_n, const int32_t* n_epj_of, const int32_t* n_spj_of, Plan& pl) {
    pl.list_off.assign((size_t)n_group + 1, 0);
    pl.inter.assign((size_t)n_group + 1, 0);
    for (int64_t g = 0; g < n_group; ++g) {
        const int64_t n_list = (int64_t)n_epj_of[g] + n_spj_of[g];
        const int64_t n_tiles = ((int64_t)n_epj_of[g] + TILE_J - 1) / TILE_J + ((int64_t)n_spj_of[g] + TILE_J - 1) / TILE_J;  // each run in whole tiles
        pl.list_off[(size_t)g + 1] = pl.list_off[(size_t)g] + n_tiles * TILE_J;
        pl.inter[(size_t)g + 1] = pl.inter[(size_t)g] + (int64_t)grp_n[g] * n_list;
    }
    // The group ranges that mwf_calc_force_all dispatches per tag for a host destination, by interaction count: equal
    // shares for the first half of the tags, then tapering to an eighth of a share.  The tags finish in order (stream
    // priorities), the copies of tag t hide behind the kernels of the tags after it, and what nothing hides -- the D2H
    // (and, in the pipelined loop, the H2D) of the LAST tag -- shrinks with its share.
    const int n_tag = c->p.n_tag;
    pl.split.assign((size_t)n_tag + 1, 0);
    const int64_t total = pl.inter[(size_t)n_group];
    std::vector<double> share((size_t)n_tag);
    double sum = 0.0;
    for (int t = 0; t < n_tag; ++t) sum += share[(size_t)t] = MWF_TAPER ? std::min(1.0, 2.0 * (n_tag - t - 0.5) / n_tag) : 1.0;
    int64_t g = 0;
    double acc = 0.0;
    for (int t = 1; t < n_tag; ++t) {
        acc += share[(size_t)t - 1];
        const int64_t want = (int64_t)((double)total * (acc / sum));
        while (g < n_group && pl.inter[(size_t)g] < want) ++g;
        pl.split[(size_t)t] = g;
    }
    pl.split[(size_t)n_tag] = n_group;
    return MWF_OK;
}

int make_plan(mwf_ctx* c, int64_t n_group, const int32_t* grp_first, const int32_t* grp_n, const int32_t* n_epj_of, const int32_t* n_spj_of, Plan& pl) {
    int rc = plan_cut(c, n_group, grp_first, grp_n, pl);
    if (rc) return rc;
    return plan_finish(c, n_group, grp_n, n_epj_of, n_spj_of, pl);
}

// Adopt a plan as the ctx's current lists (after the device side is in place).
void adopt_plan(mwf_ctx* c, Plan& pl, int64_t n_group, const int32_t* grp_first, const int32_t* grp_n, int mode) {
    c->n_items = (int64_t)pl.items.size();
    c->padded_entries = pl.list_off[(size_t)n_group];
    c->h_item_off.swap(pl.item_off);
    c->h_inter.swap(pl.inter);
    c->h_split.swap(pl.split);
    c->h_items.swap(pl.items);
    c->cls_ready = false;
    c->split_ready = false;
    c->h_grp_first.assign(grp_first, grp_first + n_group);
    c->h_grp_n.assign(grp_n, grp_n + n_group);
    c->n_group = n_group;
    c->have_lists = true;
    c->lists_for_reuse = (mode == MWF_MAKE_LIST_FOR_REUSE);
    c->groups_dispatched = 0;
    c->groups_outstanding = 0;
}

// The schedule over everything (sched_kernel.cu).  A store that does not fit the L2 is walked in SCHED_WINDOWS windows of
// consecutive (Morton-ordered) items of equal modelled cost: the gathers of the items in flight then touch one stretch of
// the store at a time (config 4, 171 MB store: DRAM traffic 6.7 -> 3.1 GB per launch at the same kernel time; a store that
// fits loses 0.3-0.7 % to the less even mix of long and short items, so it keeps one window).
int schedule_full(mwf_ctx* c, int64_t n_items, cudaStream_t s) {
    const int64_t store_bytes = (c->n_ptcl + c->n_cell + 1) * (int64_t)sizeof(float4);
    SchedTags none{};
    CU(c, launch_schedule(c->sched, c->items, n_items, c->list_off, store_bytes > c->l2_bytes ? SCHED_WINDOWS : 1, none, c->order_full, s));
    c->n_launch += 8;
    return MWF_OK;
}

// Per-tag schedules: made the first time a dispatch covers exactly one of the balanced ranges.
int ensure_split_order(mwf_ctx* c, cudaStream_t s) {
    if (c->split_ready) return MWF_OK;
    SchedTags tags{};
    tags.n_tag = c->p.n_tag;
    for (int t = 0; t <= c->p.n_tag; ++t) tags.bound[t] = (int32_t)c->h_split[(size_t)t];
    CU(c, launch_schedule(c->sched, c->items, c->n_items, c->list_off, 1, tags, c->order_split, s));
    CU(c, cudaStreamSynchronize(s));  // the other tags' streams read it too
    c->n_launch += 8;
    c->split_ready = true;
    return MWF_OK;
}

}  // namespace mwf
