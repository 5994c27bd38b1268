// Entry points of the SURVEY.md section 8(f) rows: device-resident integration (NEXT-1), quadrupole SPJ (NEXT-3),
// short-range workload (NEXT-4).
#include "mwf_ctx.h"

using namespace mwf;

static int integrate_ready(mwf_ctx* c, float dt) {
    if (!c || !(dt == dt)) return MWF_EINVAL;
    if (!c->have_tree || !c->have_lists || !c->acc_full || c->vel_hi < c->n_ptcl) return MWF_ESTATE;
    return MWF_OK;
}

static int sph_dispatch(mwf_ctx* c, int32_t tag, int64_t g_begin, int64_t g_end, bool hydro, float gamma) {
    if (!c || tag < 0 || tag >= c->p.n_tag || g_begin < 0 || g_end < g_begin) return MWF_EINVAL;
    if (!hydro && !(gamma > 1.f)) return MWF_EINVAL;
    if (!c->have_tree || !c->have_lists || !c->sph || c->sph_hi < c->n_ptcl || c->ptcl_hi < c->n_ptcl) return MWF_ESTATE;
    if (c->build_e_spj > 0) return MWF_ESTATE;  // gravity lists: their SPJ entries are monopoles, not gas particles
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
    book_dispatch(c, tag, g_begin, g_end);
    return MWF_OK;
}

extern "C" {

int mwf_set_velocities(mwf_ctx* c, const mwf_vel* src, int64_t first, int64_t n, int src_on_device, void* stream) {
    MWF_ENTER(c);
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
    MWF_ENTER(c);
    if (!c || !dst || first < 0 || n < 0 || first + n > c->p.max_ptcl) return MWF_EINVAL;
    CU(c, cudaDeviceSynchronize());
    CU(c, cudaMemcpy(dst, c->vel + first, (size_t)n * 16, dst_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost));
    return MWF_OK;
}

int mwf_kick_drift(mwf_ctx* c, float dt, void* stream) {
    MWF_ENTER(c);
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
    MWF_ENTER(c);
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
    MWF_ENTER(c);
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
    c->fuse_kick_h = 0.5f * dt;  // the closing kick rides in the force kernel's epilogue
    rc = mwf_dispatch(c, 0, 0, c->n_group);
    c->fuse_kick_h = 0.f;
    return rc;
}

// ---- short-range workload (NEXT-4)

int mwf_set_sph(mwf_ctx* c, const mwf_sph* src, int64_t first, int64_t n, int src_on_device, void* stream) {
    MWF_ENTER(c);
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
    MWF_ENTER(c);
    if (!c || !dst || first < 0 || n < 0) return MWF_EINVAL;
    if (!c->sph || first + n > c->sph_hi) return MWF_ESTATE;
    CU(c, cudaDeviceSynchronize());
    CU(c, cudaMemcpy(dst, c->sph + first, (size_t)n * 16, dst_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost));
    return MWF_OK;
}

int mwf_dispatch_density(mwf_ctx* c, int32_t tag, int64_t g_begin, int64_t g_end, float gamma) {
    MWF_ENTER(c);
    return sph_dispatch(c, tag, g_begin, g_end, false, gamma);
}

int mwf_dispatch_hydro(mwf_ctx* c, int32_t tag, int64_t g_begin, int64_t g_end) {
    MWF_ENTER(c);
    return sph_dispatch(c, tag, g_begin, g_end, true, 0.f);
}

int mwf_calc_sph_all(mwf_ctx* c, const mwf_posm* src, int src_on_device, mwf_sph* rec, int rec_on_device, mwf_accp* dst, int dst_on_device, float gamma) {
    MWF_ENTER(c);
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
    MWF_ENTER(c);
    if (!c || (order != 1 && order != 2)) return MWF_EINVAL;
    for (int t = 0; t < c->p.n_tag; ++t)
        if (c->tag_inflight[t] || !c->tag_ranges[t].empty()) return MWF_ESTATE;
    if (order == 2 && !c->quad) {
        // first the shared-memory opt-in of the order-2 kernel on this ctx's device and its occupancy; the arrays only once
        // that has succeeded, so that a failed call leaves the ctx at order 1 with nothing half set up
        const int ctas = force_quad_max_ctas_per_sm();
        if (ctas < 1) return cuda_fail(c, cudaGetLastError(), "order-2 force kernel: shared-memory opt-in / occupancy");
        void *a = nullptr, *b = nullptr;
        if (cudaMalloc(&a, (size_t)c->p.max_cell * 48) != cudaSuccess || cudaMalloc(&b, (size_t)c->p.max_cell * 32) != cudaSuccess) {
            cudaGetLastError();
            if (a) cudaFree(a);
            return MWF_ENOMEM;
        }
        c->quad64 = static_cast<double*>(a);
        c->quad = static_cast<float4*>(b);
        c->quad_ctas_per_sm = ctas;
    }
    if (order != c->spj_order) {
        c->mono_fresh = false;  // the moments on the device are those of the other order
        c->acc_full = false;
    }
    c->spj_order = order;
    return MWF_OK;
}

int mwf_get_quadrupoles(mwf_ctx* c, float* dst, int dst_on_device) {
    MWF_ENTER(c);
    if (!c || !dst) return MWF_EINVAL;
    if (!c->have_tree || !c->mono_fresh || c->spj_order != 2) return MWF_ESTATE;
    CU(c, cudaDeviceSynchronize());
    CU(c, cudaMemcpy(dst, c->quad, (size_t)c->n_cell * 32, dst_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost));
    return MWF_OK;
}

}  // extern "C"
