// Device-side construction step behind mwf_build / mwf_build_neighbours and its read-back hooks
// (SURVEY.md section 8(f) NEXT-2).
#include <cstring>

#include "mwf_ctx.h"

using namespace mwf;

// The device-side construction step behind mwf_build (opening angle theta) and mwf_build_neighbours (search radii 2 (1 + skin) h).
// The construction step failed after the particles (and velocities, SPH records) were sorted in place: what the store
// holds is a permutation the caller cannot name, so it counts as not uploaded (the caller uploads again before retrying).
static int build_failed(mwf_ctx* c, cudaStream_t s, int code) {
    after_store_op(c, s);
    c->ptcl_hi = c->vel_hi = c->sph_hi = 0;
    c->cls_hi = 0;
    c->n_ptcl = 0;
    return code;
}

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
    if (n_cell > c->p.max_cell || n_group > c->p.max_group) return build_failed(c, s, MWF_ENOMEM);
    // Everything up to the counting walk is enqueued without a host synchronisation; small results travel to pinned host
    // memory on the stream.  The group ranges come first, so that the host cuts the groups into work items while the
    // device ranks the leaves and walks the tree.
    const auto D2H = cudaMemcpyDeviceToHost;
    int32_t *h_first = c->h_groups, *h_n = h_first + n_group, *h_ne = h_n + n_group, *h_ns = h_ne + n_group, *h_nf = h_ns + n_group;
    int64_t* totals = c->h_scalars;                                          // [0..2] padded, EPJ, SPJ entries
    int32_t* n_leaf_pinned = reinterpret_cast<int32_t*>(c->h_scalars + 4);
    unsigned int* err_pinned = reinterpret_cast<unsigned int*>(c->h_scalars + 5);
    CU(c, cudaMemcpyAsync(h_first, c->grp_first, (size_t)n_group * 4, D2H, s));
    CU(c, cudaMemcpyAsync(h_n, c->grp_n, (size_t)n_group * 4, D2H, s));
    CU(c, cudaEventRecord(c->ev_groups, s));
    // tree state as mwf_set_tree leaves it: arrival counters zero, leaves ranked, dummy record behind the SPJ block
    CU(c, cudaMemsetAsync(c->arrive, 0, (size_t)n_cell * 4, s));
    CU(c, launch_leaf_ranking(c->cells, n_cell, n, c->bb.mark, c->bb.scan_scratch, c->cell_lr, n_leaf_pinned, s));
    c->n_launch += 5;
    CU(c, cudaMemsetAsync(c->store + n + n_cell, 0, 16, s));
    CU(c, cudaMemsetAsync(c->store_next + n + n_cell, 0, 16, s));
    CU(c, cudaMemsetAsync(c->spj_lo + n_cell, 0, 16, s));
    c->next_ranges.clear();
    c->next_streams.clear();
    c->n_ptcl = n;
    c->n_cell = n_cell;
    c->ptcl_hi = n;
    c->cls_hi = n;  // the store is in the order of the tree just built
    // lists: counting walk, offsets, capacity check, fill walk
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
    CU(c, build_lists_count(c->bb, n_group, rule, c->walk_warps_n, totals, s));
    CU(c, cudaMemcpyAsync(h_ne, c->bb.n_epj, (size_t)n_group * 4, D2H, s));
    CU(c, cudaMemcpyAsync(h_ns, c->bb.n_spj, (size_t)n_group * 4, D2H, s));
    CU(c, cudaMemcpyAsync(h_nf, c->bb.n_far, (size_t)n_group * 4, D2H, s));
    CU(c, cudaMemcpyAsync(err_pinned, c->err, sizeof(unsigned int), D2H, s));
    // host, meanwhile: the work items
    Plan plan;
    CU(c, cudaEventSynchronize(c->ev_groups));
    rc = plan_cut(c, n_group, h_first, h_n, plan);
    tm.lap("host: cutting | leaf ranking + counting walk");
    CU(c, cudaStreamSynchronize(s));
    tm.lap("counting walk: rest");
    c->n_leaf_cells = *n_leaf_pinned;
    if (rc) return build_failed(c, s, rc);
    if (*err_pinned) return build_failed(c, s, MWF_ENOMEM);
    const int64_t padded = totals[0], e_epj = totals[1], e_spj = totals[2];
    if (e_epj + e_spj > c->p.max_entry) return build_failed(c, s, MWF_ENOMEM);
    CU(c, build_lists_fill(c->bb, n_group, rule, c->walk_warps_n, n, n_cell, s));
    CU(c, cudaMemsetAsync(c->grp_self, 1, (size_t)n_group, s));  // theta <= 1: a group's own cells are always opened
    c->n_launch += 6;
    // beside the fill walk, on a stream of its own: the work items go up and are scheduled (the list offsets they need were
    // made by the counting pass, which the host has just waited for)
    const int64_t n_items = (int64_t)plan.items.size();
    CU(c, cudaMemcpyAsync(c->items, plan.items.data(), (size_t)n_items * sizeof(WorkItem), cudaMemcpyHostToDevice, c->aux_stream));
    rc = schedule_full(c, n_items, c->aux_stream);
    if (rc) return build_failed(c, s, rc);
    // host, meanwhile: list offsets and interaction counts per group, the tags' group ranges
    CU(c, cudaEventRecord(c->ev_aux, c->aux_stream));
    CU(c, cudaStreamWaitEvent(s, c->ev_aux, 0));
    for (int64_t g = 0; g < n_group; ++g) {  // the two runs of every list: EPJ + far SPJ, near SPJ
        h_ne[g] += h_nf[g];
        h_ns[g] -= h_nf[g];
    }
    rc = plan_finish(c, n_group, h_n, h_ne, h_ns, plan);
    tm.lap("host: offsets | fill walk, schedule");
    if (rc) return build_failed(c, s, rc);
    if (plan.list_off[(size_t)n_group] != padded) return build_failed(c, s, MWF_ERANGE);  // host and device offsets must agree
    CU(c, cudaStreamSynchronize(s));  // the plan's host vectors die with this call
    tm.lap("fill walk, schedule: rest");
    rc = after_store_op(c, s);
    if (rc) return rc;
    c->have_tree = true;
    c->built_on_device = true;
    c->build_e_epj = e_epj;
    c->build_e_spj = e_spj;
    c->build_n_level = n_level;
    adopt_plan(c, plan, n_group, h_first, h_n, mode);
    return MWF_OK;
}

extern "C" {

int mwf_build(mwf_ctx* c, int64_t n, int32_t n_leaf, int32_t n_grp, double theta, int mode, void* stream) {
    MWF_ENTER(c);
    return build_impl(c, n, n_leaf, n_grp, theta, false, 0.0, mode, stream);
}

int mwf_build_neighbours(mwf_ctx* c, int64_t n, int32_t n_leaf, int32_t n_grp, double skin, int mode, void* stream) {
    MWF_ENTER(c);
    return build_impl(c, n, n_leaf, n_grp, 0.0, true, skin, mode, stream);
}

int mwf_get_build_sizes(mwf_ctx* c, int64_t* n_cell, int64_t* n_group, int64_t* n_epj, int64_t* n_spj, int32_t* n_level) {
    MWF_ENTER(c);
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
    MWF_ENTER(c);
    if (!c || !perm) return MWF_EINVAL;
    if (!c->built_on_device) return MWF_ESTATE;
    CU(c, cudaDeviceSynchronize());
    CU(c, cudaMemcpy(perm, c->bb.idx_a, (size_t)c->n_ptcl * 4, dst_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost));
    return MWF_OK;
}

int mwf_get_tree(mwf_ctx* c, mwf_cell* cells, double* geom4) {
    MWF_ENTER(c);
    if (!c || (!cells && !geom4)) return MWF_EINVAL;
    if (!c->have_tree) return MWF_ESTATE;
    if (geom4 && !c->built_on_device) return MWF_ESTATE;  // an uploaded tree carries no geometry
    CU(c, cudaDeviceSynchronize());
    if (cells) CU(c, cudaMemcpy(cells, c->cells, (size_t)c->n_cell * sizeof(mwf_cell), cudaMemcpyDeviceToHost));
    if (geom4) CU(c, cudaMemcpy(geom4, c->bb.geom, (size_t)c->n_cell * 32, cudaMemcpyDeviceToHost));
    return MWF_OK;
}

int mwf_get_groups(mwf_ctx* c, int32_t* grp_first, int32_t* grp_n) {
    MWF_ENTER(c);
    if (!c || !grp_first || !grp_n) return MWF_EINVAL;
    if (!c->have_lists) return MWF_ESTATE;
    std::memcpy(grp_first, c->h_grp_first.data(), (size_t)c->n_group * 4);
    std::memcpy(grp_n, c->h_grp_n.data(), (size_t)c->n_group * 4);
    return MWF_OK;
}

int mwf_get_lists(mwf_ctx* c, int64_t* epj_off, int32_t* epj_id, int64_t* spj_off, int32_t* spj_id) {
    MWF_ENTER(c);
    if (!c || !epj_off || !spj_off || !epj_id || !spj_id) return MWF_EINVAL;
    if (!c->have_lists) return MWF_ESTATE;
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

int mwf_get_list_buffer(mwf_ctx* c, int64_t* list_off, int32_t* list, int64_t* n_group, int64_t* n_entry, int dst_on_device) {
    MWF_ENTER(c);
    if (!c) return MWF_EINVAL;
    if (!c->have_lists) return MWF_ESTATE;
    if (n_group) *n_group = c->n_group;
    if (n_entry) *n_entry = c->padded_entries;
    CU(c, cudaDeviceSynchronize());
    const auto kind = dst_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
    if (list_off) CU(c, cudaMemcpy(list_off, c->list_off, (size_t)(c->n_group + 1) * 8, kind));
    if (list && c->padded_entries > 0) CU(c, cudaMemcpy(list, c->list, (size_t)c->padded_entries * 4, kind));
    return MWF_OK;
}

int mwf_get_run1_len(mwf_ctx* c, int32_t* run1_len, int dst_on_device) {
    MWF_ENTER(c);
    if (!c || !run1_len) return MWF_EINVAL;
    if (!c->have_lists) return MWF_ESTATE;
    CU(c, cudaDeviceSynchronize());
    CU(c, cudaMemcpy(run1_len, c->grp_run1, (size_t)c->n_group * 4, dst_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost));
    return MWF_OK;
}

}  // extern "C"
