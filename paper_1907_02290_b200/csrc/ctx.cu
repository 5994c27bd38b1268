// Context of libmwf.so: arena layout, creation / destruction, stream and event plumbing, error texts
// (the C ABI of include/mwf.h).
#include <cstring>
#include <new>

#include "mwf_ctx.h"
#include "scan_sort.cuh"

using namespace mwf;

namespace mwf {

bool trace_on() {
    static const bool on = [] { const char* e = std::getenv("MWF_TRACE"); return e && e[0] && e[0] != '0'; }();
    return on;
}

int cuda_fail(mwf_ctx* c, cudaError_t e, const char* what) {
    if (c) {
        char buf[256];
        snprintf(buf, sizeof buf, "%s: %s", what, cudaGetErrorString(e));
        c->cuda_err = buf;
    }
    return MWF_ECUDA;
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

// MWF_REFRESH=climb in the environment: the bottom-up climb also for monopoles (A/B switch for the scan variant)
bool use_scan_refresh() {
    static const bool on = [] { const char* e = std::getenv("MWF_REFRESH"); return !(e && e[0] == 'c'); }();
    return on;
}

}  // namespace mwf

namespace {

inline int64_t up(int64_t x, int64_t a) { return (x + a - 1) / a * a; }

struct Layout {
    int64_t off[64];
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
    L.add((p.max_entry + 2 * TILE_J * p.max_group) * 4);  // 13 list (each of a group's two runs padded to whole tiles)
    L.add(mi * (int64_t)sizeof(WorkItem));              // 14 items
    L.add(mi * 4);                                      // 15 order_full
    L.add(mi * 4);                                      // 16 order_split
    L.add(N_COUNTER * 4);                               // 17 counters
    L.add(256);                                         // 18 err
    L.add(p.max_ptcl * 16);                             // 19 vel
    // device-side construction step (NEXT-2)
    const int64_t nsb = sort_blocks(std::max<int64_t>(p.max_ptcl, mi));  // the sort of the particles' keys and that of the work items' share the scratch
    const int64_t scan_n = std::max<int64_t>(std::max<int64_t>(256 * nsb + 1, p.max_ptcl + 2), p.max_cell + 2);
    L.add(p.max_ptcl * 8);                              // 20 key_a
    L.add(p.max_ptcl * 8);                              // 21 key_b
    L.add(p.max_ptcl * 4);                              // 22 idx_a (the permutation after a build)
    L.add(p.max_ptcl * 4);                              // 23 idx_b
    L.add((256 * nsb + 1) * 4);                         // 24 hist
    L.add(scan_scratch_elems(scan_n) * 4);              // 25 scan_scratch (int32)
    L.add(scan_scratch_elems(std::max<int64_t>(p.max_group + 2, mi + 2)) * 8);  // 26 scan_scratch64
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
    L.add((p.max_cell + 1) * 16);                       // 43 spj_lo
    L.add(p.max_group * 4);                             // 44 grp_nfar
    L.add(p.max_group * 4);                             // 45 grp_run1
    L.add((mi + 1) * 8);                                // 46 sched cost
    L.add((mi + 1) * 8);                                // 47 sched cum
    L.add(mi * 8);                                      // 48 sched key_a
    L.add(mi * 8);                                      // 49 sched key_b
    L.add(mi * 4);                                      // 50 sched idx_a
    L.add(mi * 4);                                      // 51 sched idx_b
    L.add(256);                                         // 52 sched seg (2 x max(SCHED_WINDOWS, MWF_MAX_TAG) + 1 ints)
    L.add(mi * 4);                                      // 53 order_cls
    return L;
}

bool params_ok(const mwf_params* p) {
    if (!p) return false;
    if (!(p->eps > 0.f) || !(p->eps * p->eps >= 1.17549435e-38f)) return false;
    if (!(p->G == p->G)) return false;
    if (p->max_ptcl < 1 || p->max_cell < 1 || p->max_group < 1 || p->max_entry < 1) return false;
    if (p->max_ptcl + p->max_cell + 1 > 0x7fffffffLL) return false;  // 32-bit list indices
    if (p->max_cell >= 0x40000000LL) return false;                   // one bit of a cell index is borrowed while lists are re-encoded
    if (p->n_tag < 1 || p->n_tag > MWF_MAX_TAG) return false;
    if (p->device < 0) return false;
    return true;
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

const char* mwf_last_cuda_error(mwf_ctx* c) {
    MWF_ENTER(c); return c ? c->cuda_err.c_str() : ""; }

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
    c->spj_lo = (float4*)(b + L.off[43]);
    c->grp_nfar = (int32_t*)(b + L.off[44]);
    c->grp_run1 = (int32_t*)(b + L.off[45]);
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
    c->order_cls = (int32_t*)(b + L.off[53]);
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
        q.n_far = c->grp_nfar; q.run1_len = c->grp_run1;
        q.list_off = c->list_off; q.epj_off = c->st_epj_off; q.spj_off = c->st_spj_off; q.list = c->list;
        q.walk_stacks = (int32_t*)(b + L.off[36]); q.walk_counter = (unsigned int*)(b + L.off[37]); q.err = c->err;
        q.level_bounds = (int32_t*)(b + L.off[38]);
        c->walk_warps_n = walk_warps(p->max_group);
    }
    c->sched.cost = (int64_t*)(b + L.off[46]); c->sched.cum = (int64_t*)(b + L.off[47]);
    c->sched.key_a = (uint64_t*)(b + L.off[48]); c->sched.key_b = (uint64_t*)(b + L.off[49]);
    c->sched.idx_a = (int32_t*)(b + L.off[50]); c->sched.idx_b = (int32_t*)(b + L.off[51]);
    c->sched.seg = (int32_t*)(b + L.off[52]);
    c->sched.hist = c->bb.hist; c->sched.scan_scratch = c->bb.scan_scratch; c->sched.scan_scratch64 = c->bb.scan_scratch64;
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
    }
    ok = ok && cudaEventCreateWithFlags(&c->ev_store, cudaEventDisableTiming) == cudaSuccess;
    ok = ok && cudaEventCreateWithFlags(&c->ev_next, cudaEventDisableTiming) == cudaSuccess;
    ok = ok && cudaMemset(c->counters, 0, N_COUNTER * 4) == cudaSuccess;
    ok = ok && cudaMemset(c->err, 0, 256) == cudaSuccess;
    ok = ok && cudaHostAlloc(reinterpret_cast<void**>(&c->h_scalars), 16 * sizeof(int64_t), cudaHostAllocDefault) == cudaSuccess;
    c->bb.h_i32 = ok ? reinterpret_cast<int32_t*>(c->h_scalars + 8) : nullptr;
    ok = ok && cudaHostAlloc(reinterpret_cast<void**>(&c->h_order_cls), (size_t)c->max_items * sizeof(int32_t), cudaHostAllocDefault) == cudaSuccess;
    ok = ok && cudaHostAlloc(reinterpret_cast<void**>(&c->h_groups), (size_t)p->max_group * 5 * sizeof(int32_t), cudaHostAllocDefault) == cudaSuccess;
    ok = ok && cudaEventCreateWithFlags(&c->ev_groups, cudaEventDisableTiming) == cudaSuccess;
    ok = ok && cudaStreamCreateWithFlags(&c->aux_stream, cudaStreamNonBlocking) == cudaSuccess;
    ok = ok && cudaEventCreateWithFlags(&c->ev_aux, cudaEventDisableTiming) == cudaSuccess;
    if (!ok) { mwf_destroy(c); return MWF_ECUDA; }
    *out = c;
    return MWF_OK;
}

int mwf_destroy(mwf_ctx* c) {
    MWF_ENTER(c);
    if (c && c->sph) { cudaFree(c->sph); c->sph = nullptr; }
    if (!c) return MWF_EINVAL;
    cudaDeviceSynchronize();
    for (int t = 0; t < MWF_MAX_TAG; ++t) {
        if (c->tag_own[t] && c->tag_stream[t]) cudaStreamDestroy(c->tag_stream[t]);
        if (c->ev_tag[t]) cudaEventDestroy(c->ev_tag[t]);
        if (c->ev_k0[t]) cudaEventDestroy(c->ev_k0[t]);
        if (c->ev_k1[t]) cudaEventDestroy(c->ev_k1[t]);
    }
    if (c->h_scalars) cudaFreeHost(c->h_scalars);
    if (c->h_groups) cudaFreeHost(c->h_groups);
    if (c->h_order_cls) cudaFreeHost(c->h_order_cls);
    if (c->ev_groups) cudaEventDestroy(c->ev_groups);
    if (c->aux_stream) cudaStreamDestroy(c->aux_stream);
    if (c->ev_aux) cudaEventDestroy(c->ev_aux);
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
    MWF_ENTER(c);
    if (!c || tag < 0 || tag >= c->p.n_tag) return MWF_EINVAL;
    if (c->tag_inflight[tag] || !c->tag_ranges[tag].empty()) return MWF_ESTATE;
    if (c->tag_own[tag] && c->tag_stream[tag]) cudaStreamDestroy(c->tag_stream[tag]);
    c->tag_own[tag] = false;
    c->tag_stream[tag] = static_cast<cudaStream_t>(cuda_stream);
    return MWF_OK;
}

int mwf_device_pointers(mwf_ctx* c, mwf_posm** store, mwf_accp** accp) {
    MWF_ENTER(c);
    if (!c) return MWF_EINVAL;
    if (store) *store = reinterpret_cast<mwf_posm*>(c->store);
    if (accp) *accp = reinterpret_cast<mwf_accp*>(c->accp);
    return MWF_OK;
}

int mwf_sync(mwf_ctx* c) {
    MWF_ENTER(c);
    if (!c) return MWF_EINVAL;
    CU(c, cudaDeviceSynchronize());
    return MWF_OK;
}

int mwf_get_counters(mwf_ctx* c, int64_t* kernel_launches, int64_t* interactions, int64_t* padded_entries) {
    MWF_ENTER(c);
    if (!c) return MWF_EINVAL;
    if (kernel_launches) *kernel_launches = c->n_launch;
    if (interactions) *interactions = c->n_inter;
    if (padded_entries) *padded_entries = c->padded_entries;
    return MWF_OK;
}

}  // extern "C"
