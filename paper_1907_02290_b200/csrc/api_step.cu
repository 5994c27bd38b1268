// The five calls of the hot path and the list-reuse driver:
// particles, tree, lists, refresh, dispatch, retrieve.
#include <cstring>

#include "mwf_ctx.h"

using namespace mwf;

namespace mwf {

// The schedule of a dispatch over groups [g_begin, g_end): the full one, a per-tag one, or none (item order).
int pick_order(mwf_ctx* c, int64_t g_begin, int64_t g_end, cudaStream_t s, const int32_t** order) {
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
void book_dispatch(mwf_ctx* c, int32_t tag, int64_t g_begin, int64_t g_end) {
    c->tag_inflight[tag] = true;
    c->cls_hi = 0;  // the store has been used with the current tree: uploads from here on are the next step's
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

}  // namespace mwf

// Launch of the force kernel over groups [g_begin, g_end) on the tag's stream and the bookkeeping that goes with it.
// jdata / joff (device) non-null: method G1, the lists are runs of j records instead of indices into the store.
static int dispatch_launch(mwf_ctx* c, int32_t tag, int64_t g_begin, int64_t g_end, const float4* jdata, const int64_t* joff) {
    cudaStream_t s = c->tag_stream[tag];
    ForceArgs a;
    a.store = c->store;
    a.spj_lo = c->spj_lo;
    a.n_ptcl = (int32_t)c->n_ptcl;
    a.dummy = (int32_t)(c->n_ptcl + c->n_cell);
    a.run1_len = c->grp_run1;
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
    a.quad = (c->spj_order == 2 && !jdata) ? c->quad : nullptr;  // order 2: the Q terms of the SPJ entries in the same sweep
    a.n_far = c->grp_nfar;
    a.n_cell = (int32_t)c->n_cell;
    a.vel = (c->fuse_kick_h != 0.f && !jdata) ? c->vel : nullptr;
    a.kick_h = c->fuse_kick_h;
    {
        const int rc = pick_order(c, g_begin, g_end, s, &a.order);
        if (rc) return rc;
    }
    a.n_seg = 0;
    if (!a.order && !jdata) {  // any other group range: its items widest first, from the class-sorted permutation
        const int rc = ensure_class_order(c, s);
        if (rc) return rc;
        a.order = c->order_cls;
        a.n_seg = N_WIDTH_CLASS;
        a.seg_cum[0] = 0;
        for (int k = 0; k < N_WIDTH_CLASS; ++k) {
            const int64_t lo = c->h_cls_off[k][(size_t)g_begin], hi = c->h_cls_off[k][(size_t)g_end];
            a.seg_begin[k] = c->h_cls_base[k] + lo;
            a.seg_cum[k + 1] = a.seg_cum[k] + (hi - lo);
        }
    }
    const int64_t resident = (int64_t)c->n_sm * (a.quad ? c->quad_ctas_per_sm : c->ctas_per_sm);
    if (resident < 1) return cuda_fail(c, cudaErrorLaunchOutOfResources, "force kernel: no block fits an SM");  // never a silent empty launch
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
    CU(c, cudaEventRecord(c->ev_k1[tag], s));
    CU(c, cudaEventRecord(c->ev_tag[tag], s));
    c->tag_timed[tag] = true;
    book_dispatch(c, tag, g_begin, g_end);
    c->groups_dispatched += g_end - g_begin;
    if (c->groups_dispatched >= c->n_group) c->acc_full = true;
    return MWF_OK;
}

extern "C" {

int mwf_set_particles(mwf_ctx* c, const mwf_posm* src, int64_t first, int64_t n, int src_on_device, void* stream) {
    MWF_ENTER(c);
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
    if (first <= c->cls_hi) c->cls_hi = std::max(c->cls_hi, first + n);
    c->mono_fresh = false;
    c->acc_full = false;
    return after_store_op(c, s);
}

int mwf_set_particles_next(mwf_ctx* c, const mwf_posm* src, int64_t first, int64_t n, int src_on_device, void* stream) {
    MWF_ENTER(c);
    if (!c || !src || first < 0 || n < 0) return MWF_EINVAL;
    if (!c->have_tree) return MWF_ESTATE;
    if (first + n > c->n_ptcl) return MWF_ERANGE;
    if (n == 0) return MWF_OK;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    // no kernel reads the shadow store (its last readers were retrieved before the swap that made it the shadow), but an
    // asynchronous mwf_set_particles into what was then the store may still be writing it
    if (c->store_event_valid) CU(c, cudaStreamWaitEvent(s, c->ev_store, 0));
    CU(c, cudaMemcpyAsync(c->store_next + first, src, (size_t)n * 16, src_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, s));
    c->next_ranges.emplace_back(first, first + n);
    if (std::find(c->next_streams.begin(), c->next_streams.end(), s) == c->next_streams.end()) c->next_streams.push_back(s);
    return MWF_OK;
}

int mwf_swap_store(mwf_ctx* c, void* stream) {
    MWF_ENTER(c);
    if (!c) return MWF_EINVAL;
    if (!c->have_tree) return MWF_ESTATE;
    {   // the uploads since the last swap must tile [0, N) exactly: a hole would keep positions from two steps back
        auto& r = c->next_ranges;
        std::sort(r.begin(), r.end());
        int64_t at = 0;
        for (const auto& q : r) {
            if (q.first != at) return MWF_ESTATE;
            at = q.second;
        }
        if (at != c->n_ptcl) return MWF_ESTATE;
    }
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
    c->next_ranges.clear();
    c->next_streams.clear();
    c->ptcl_hi = c->n_ptcl;
    c->cls_hi = c->n_ptcl;
    c->mono_fresh = false;
    c->acc_full = false;
    return after_store_op(c, s);  // every later dispatch / store operation waits for this event, hence for the uploads
}

int mwf_get_tag_split(mwf_ctx* c, int64_t* bounds) {
    MWF_ENTER(c);
    if (!c || !bounds) return MWF_EINVAL;
    if (!c->have_lists) return MWF_ESTATE;
    for (int t = 0; t <= c->p.n_tag; ++t) bounds[t] = c->h_split[(size_t)t];
    return MWF_OK;
}

int mwf_get_particles(mwf_ctx* c, mwf_posm* dst, int64_t first, int64_t n, int dst_on_device) {
    MWF_ENTER(c);
    if (!c || !dst || first < 0 || n < 0) return MWF_EINVAL;
    if (first + n > (c->have_tree ? c->n_ptcl : c->ptcl_hi)) return MWF_ERANGE;  // behind the particles: SPJ block / unwritten store
    CU(c, cudaDeviceSynchronize());
    CU(c, cudaMemcpy(dst, c->store + first, (size_t)n * 16, dst_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost));
    return MWF_OK;
}

int mwf_set_tree(mwf_ctx* c, const mwf_cell* cells, int64_t n_cell, void* stream) {
    MWF_ENTER(c);
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
    c->n_launch += 2;
    {   // a tree that failed the validation must not be ranked (its ranges may point anywhere)
        unsigned int e0 = 0;
        rc = read_err_word(c, s, &e0);
        if (rc) return rc;
        if (e0) { after_store_op(c, s); return MWF_ERANGE; }
    }
    int32_t* n_leaf_pinned = reinterpret_cast<int32_t*>(c->h_scalars);
    CU(c, launch_leaf_ranking(c->cells, n_cell, n, c->bb.mark, c->bb.scan_scratch, c->cell_lr, n_leaf_pinned, s));
    c->n_launch += 5;
    // zero-mass dummy record behind the SPJ block: what list padding points at
    const float4 zero = make_float4(0.f, 0.f, 0.f, 0.f);
    CU(c, cudaMemcpyAsync(c->store + n + n_cell, &zero, 16, cudaMemcpyHostToDevice, s));
    CU(c, cudaMemcpyAsync(c->store_next + n + n_cell, &zero, 16, cudaMemcpyHostToDevice, s));
    CU(c, cudaMemsetAsync(c->spj_lo + n_cell, 0, 16, s));
    c->next_ranges.clear();
    c->next_streams.clear();
    unsigned int e = 0;
    rc = read_err_word(c, s, &e);  // synchronises the stream: the number of leaves has arrived too
    if (rc) return rc;
    c->n_leaf_cells = *n_leaf_pinned;
    rc = after_store_op(c, s);
    if (rc) return rc;
    if (e) return MWF_ERANGE;
    c->n_ptcl = n;
    c->n_cell = n_cell;
    c->ptcl_hi = std::min(c->ptcl_hi, n);
    c->cls_hi = std::min(c->cls_hi, n);
    c->have_tree = true;
    return MWF_OK;
}

int mwf_set_lists(mwf_ctx* c, int64_t n_group, const int32_t* grp_first, const int32_t* grp_n, const int64_t* epj_off,
                  const int32_t* epj_id, const int64_t* spj_off, const int32_t* spj_id, int mode, void* stream) {
    MWF_ENTER(c);
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
    std::vector<int32_t> n_epj((size_t)n_group), n_spj((size_t)n_group);
    for (int64_t g = 0; g < n_group; ++g) {
        const int64_t ne = epj_off[g + 1] - epj_off[g], ns = spj_off[g + 1] - spj_off[g];
        if (ne < 0 || ns < 0 || ne > INT32_MAX || ns > INT32_MAX) return MWF_ERANGE;
        n_epj[(size_t)g] = (int32_t)ne;
        n_spj[(size_t)g] = (int32_t)ns;
    }
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
    // which SPJ entries are far enough to be swept like particles (run 1); their number per group sizes the two runs
    // (only from positions uploaded for THIS step: what an earlier step left in the store is in the previous tree's order)
    const bool have_ptcl = c->ptcl_hi >= c->n_ptcl && c->cls_hi >= c->n_ptcl;
    // (the cells' tight boxes live in mom64 for the moment: 32 B per cell, rewritten from the leaves up by every refresh that reads it)
    CU(c, launch_classify_spj(n_group, c->grp_first, c->grp_n, c->st_spj_off, c->st_ids + e_epj, c->cells, c->parent, c->arrive,
                              reinterpret_cast<float4*>(c->mom64), c->store, c->n_ptcl, c->n_cell, have_ptcl, c->grp_nfar, s));
    c->n_launch += have_ptcl ? 2 : 1;
    std::vector<int32_t> n_far((size_t)n_group);
    CU(c, cudaMemcpyAsync(n_far.data(), c->grp_nfar, (size_t)n_group * 4, cudaMemcpyDeviceToHost, s));
    CU(c, cudaStreamSynchronize(s));
    for (int64_t g = 0; g < n_group; ++g) {  // run 1 = EPJ + far SPJ, run 2 = near SPJ
        if (n_far[(size_t)g] < 0 || n_far[(size_t)g] > n_spj[(size_t)g]) { after_store_op(c, s); return cuda_fail(c, cudaErrorUnknown, "SPJ classification"); }
        n_epj[(size_t)g] += n_far[(size_t)g];
        n_spj[(size_t)g] -= n_far[(size_t)g];
    }
    if (trace_on()) {
        int64_t nf = 0;
        for (int64_t g = 0; g < n_group; ++g) nf += n_far[(size_t)g];
        fprintf(stderr, "[mwf trace] far SPJ entries: %lld of %lld\n", (long long)nf, (long long)e_spj);
    }
    // host pass: offsets, items, schedule
    Plan plan;
    {
        const int prc = make_plan(c, n_group, grp_first, grp_n, n_epj.data(), n_spj.data(), plan);
        if (prc) { after_store_op(c, s); return prc; }
    }
    const std::vector<int64_t>& list_off = plan.list_off;
    const std::vector<WorkItem>& items = plan.items;
    const int64_t n_items = (int64_t)items.size();
    CU(c, cudaMemcpyAsync(c->list_off, list_off.data(), (size_t)(n_group + 1) * 8, H2D, s));
    CU(c, cudaMemcpyAsync(c->items, items.data(), (size_t)n_items * sizeof(WorkItem), H2D, s));
    CU(c, launch_merge_lists(n_group, c->grp_first, c->grp_n, c->st_epj_off, c->st_ids, c->st_spj_off, c->st_ids + e_epj, c->list_off,
                             c->grp_nfar, c->grp_run1, c->n_ptcl, c->n_cell, c->list, c->grp_self, c->err, s));
    rc = schedule_full(c, n_items, s);
    if (rc) return rc;
    ++c->n_launch;
    unsigned int e = 0;
    rc = read_err_word(c, s, &e);  // also makes the host vectors above safe to free
    if (rc) return rc;
    rc = after_store_op(c, s);
    if (rc) return rc;
    if (e & ~ERR_SELF_MIXED) return MWF_ERANGE;
    if (e) return MWF_EINVAL;  // only the self-membership rule is violated
    adopt_plan(c, plan, n_group, grp_first, grp_n, mode);
    c->build_e_epj = e_epj;
    c->build_e_spj = e_spj;
    return MWF_OK;
}

int mwf_begin_step(mwf_ctx* c, int mode) {
    MWF_ENTER(c);
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
    MWF_ENTER(c);
    if (!c) return MWF_EINVAL;
    if (!c->have_tree || c->ptcl_hi < c->n_ptcl) return MWF_ESTATE;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    int rc = before_store_op(c, s);
    if (rc) return rc;
    if (c->spj_order == 2 || !use_scan_refresh()) {  // the quadrupoles need the bottom-up pass (parallel-axis theorem)
        CU(c, launch_monopoles(c->cells, c->parent, c->n_cell, c->n_ptcl, c->store, c->spj_lo, c->mom64, c->arrive,
                               c->spj_order == 2 ? c->quad64 : nullptr, c->spj_order == 2 ? c->quad : nullptr, s));
        ++c->n_launch;
    } else {
        CU(c, launch_monopoles_scan(c->cells, c->cell_lr, c->n_cell, c->n_ptcl, c->n_leaf_cells, c->store, c->spj_lo, c->leaf_P, c->leaf_toff, s));
        c->n_launch += 4;
    }
    c->mono_fresh = true;
    return after_store_op(c, s);
}

int mwf_dispatch(mwf_ctx* c, int32_t tag, int64_t g_begin, int64_t g_end) {
    MWF_ENTER(c);
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
    MWF_ENTER(c);
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
    MWF_ENTER(c);
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
    MWF_ENTER(c);
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
    MWF_ENTER(c);
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

int mwf_get_monopoles(mwf_ctx* c, mwf_posm* dst, int dst_on_device) {
    MWF_ENTER(c);
    if (!c || !dst) return MWF_EINVAL;
    if (!c->have_tree || !c->mono_fresh) return MWF_ESTATE;
    CU(c, cudaDeviceSynchronize());
    CU(c, cudaMemcpy(dst, c->store + c->n_ptcl, (size_t)c->n_cell * 16, dst_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost));
    return MWF_OK;
}

int mwf_last_dispatch_ms(mwf_ctx* c, int32_t tag, float* ms) {
    MWF_ENTER(c);
    if (!c || tag < 0 || tag >= c->p.n_tag || !ms) return MWF_EINVAL;
    if (!c->tag_timed[tag]) return MWF_ESTATE;
    CU(c, cudaEventSynchronize(c->ev_k1[tag]));
    CU(c, cudaEventElapsedTime(ms, c->ev_k0[tag], c->ev_k1[tag]));
    return MWF_OK;
}

}  // extern "C"
