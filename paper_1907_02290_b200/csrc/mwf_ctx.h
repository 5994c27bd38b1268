// Host-side state of one mwf_ctx and the helpers shared by the translation units that implement the C ABI
// (ctx.cu, plan.cu, api_step.cu, api_build.cu, api_next.cu).  Not part of the ABI.
#pragma once
#include <algorithm>
#include <chrono>
#include <cstdio>
#include <cstdlib>
#include <string>
#include <utility>
#include <vector>

#include "mwf_internal.h"

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
    std::vector<std::pair<int64_t, int64_t>> next_ranges;  // particle ranges written into the shadow store since the last swap
    std::vector<cudaStream_t> next_streams;  // streams those uploads went to
    float4* spj_lo = nullptr;     // [max_cell + 1] per cell: rounding remainder of the SPJ record's centre of mass (reading S11b)
    float4* accp = nullptr;       // [max_ptcl]
    float4* vel = nullptr;        // [max_ptcl] (vx, vy, vz, unused): device-resident integration
    mwf_cell* cells = nullptr;    // [max_cell]
    int32_t* parent = nullptr;    // [max_cell]
    int32_t* arrive = nullptr;    // [max_cell]
    double4* mom64 = nullptr;     // [max_cell]
    int2* cell_lr = nullptr;      // [max_cell] range of leaf ranks of every cell (scan variant of the refresh)
    double4* leaf_P = nullptr;    // [max_cell + 1] leaves' moments in rank order, scanned in place every refresh
    double4* leaf_toff = nullptr; // [tiles] scanned tile totals
    int64_t* h_scalars = nullptr; // pinned: small results of the construction step (counts, totals, validation word)
    int32_t* h_order_cls = nullptr;  // pinned [max_items]: the class-sorted permutation on its way to the device
    int32_t* h_groups = nullptr;  // pinned [5 x max_group]: group ranges and list lengths on their way to the host work plan
    cudaEvent_t ev_groups{};      // the group ranges have arrived
    cudaStream_t aux_stream{};    // construction step: the work schedule is made here while the fill walk runs on the caller's stream
    cudaEvent_t ev_aux{};
    float fuse_kick_h = 0.f;      // mwf_step_reuse: the closing kick rides in the force kernel's epilogue (0: no kick)
    int64_t n_leaf_cells = 0;
    int32_t* grp_first = nullptr; // [max_group]
    int32_t* grp_n = nullptr;     // [max_group]
    uint8_t* grp_self = nullptr;  // [max_group]
    int32_t* grp_nfar = nullptr;  // [max_group] far SPJ entries of every group (swept like particles, see SPJ_FAR_KAPPA)
    int32_t* grp_run1 = nullptr;  // [max_group] entries of run 1 = EPJ + far SPJ
    int64_t* list_off = nullptr;  // [max_group + 1]
    int64_t* st_epj_off = nullptr, *st_spj_off = nullptr;  // [max_group + 1] staging
    int32_t* st_ids = nullptr;    // [max_entry] staging of the uploaded ids
    int32_t* list = nullptr;      // [max_entry + 2 * TILE_J * max_group] merged; each of a group's two runs padded to whole tiles
    mwf::WorkItem* items = nullptr;    // [max_items]
    int32_t* order_full = nullptr, *order_split = nullptr;  // [max_items]
    // items sorted by width class (32, 16, 8, 4, 2), group order inside a class: any contiguous group range then has its
    // items widest-first as five contiguous runs (h_cls_off[k][g] = items of class k in the groups before g)
    int32_t* order_cls = nullptr;                            // [max_items]; made on first use (ensure_class_order)
    bool cls_ready = false;
    std::vector<mwf::WorkItem> h_items;                      // the work items as cut (host copy)
    std::vector<int32_t> h_cls_off[mwf::N_WIDTH_CLASS];
    int64_t h_cls_base[mwf::N_WIDTH_CLASS + 1]{};
    unsigned int* counters = nullptr;  // [N_COUNTER]
    unsigned int* err = nullptr;
    int64_t max_items = 0;
    // state
    int64_t n_ptcl = 0, n_cell = 0, n_group = 0, n_items = 0, ptcl_hi = 0, padded_entries = 0;
    bool have_tree = false, have_lists = false, lists_for_reuse = false, mono_fresh = false;
    // Particles [0, cls_hi) have been uploaded, contiguously from 0, since the last dispatch: they are the positions of the
    // step being prepared, so mwf_set_lists may classify SPJ entries as far / near from them (reading S11b).  A dispatch
    // consumes the store for the tree it ran on and resets this; when mwf_set_lists finds cls_hi < N it calls every entry near.
    int64_t cls_hi = 0;
    mwf::BuildBuffers bb{};       // device-side construction step (NEXT-2)
    int64_t walk_warps_n = 0;
    bool built_on_device = false;
    int64_t build_e_epj = 0, build_e_spj = 0;
    int32_t build_n_level = 0;
    bool acc_full = false;   // every group has been dispatched since the positions last changed
    int64_t vel_hi = 0;      // velocities [0, vel_hi) have been uploaded
    std::vector<int64_t> h_item_off, h_inter, h_split;  // per group prefix of items / interactions; split group bounds
    std::vector<int32_t> h_grp_first, h_grp_n;
    mwf::SchedBuffers sched{};            // scratch of the device-side work schedule
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
    // short-range workload (NEXT-4): per-particle SPH record, cudaMalloc'ed when mwf_set_sph() is first called
    float4* sph = nullptr;      // [max_ptcl] (h, u, rho, P/rho^2)
    int64_t sph_hi = 0;         // records [0, sph_hi) have been uploaded
    int sph_ctas_per_sm[2] = {0, 0};
    int tag_kind[MWF_MAX_TAG]{};  // what the tag's pending results are: 0 = acc/pot (or hydro acc), 1 = SPH records
    uint32_t counter_seq = 0;
    int64_t n_launch = 0, n_inter = 0;
    std::string cuda_err;
};

namespace mwf {

constexpr int N_COUNTER = 1024;

int cuda_fail(mwf_ctx* c, cudaError_t e, const char* what);
#define CU(c, call)                                                        \
    do {                                                                   \
        cudaError_t e__ = (call);                                          \
        if (e__ != cudaSuccess) return mwf::cuda_fail((c), e__, #call);    \
    } while (0)

// First statement of every entry point that takes a ctx: the calling thread may have switched device since mwf_create.
#define MWF_ENTER(c)                                   \
    do {                                               \
        if (c) cudaSetDevice((c)->p.device);           \
    } while (0)

// MWF_TRACE=1 in the environment: wall-clock phase times of the construction step on stderr
bool trace_on();
struct PhaseTimer {
    std::chrono::steady_clock::time_point t0 = std::chrono::steady_clock::now();
    void lap(const char* what) {
        if (!trace_on()) return;
        const auto t1 = std::chrono::steady_clock::now();
        fprintf(stderr, "[mwf trace] %-28s %8.3f ms\n", what, std::chrono::duration<double, std::milli>(t1 - t0).count());
        t0 = t1;
    }
};

// Every operation that writes the store / tree / lists first waits for the force kernels that read them.
int before_store_op(mwf_ctx* c, cudaStream_t s);
int after_store_op(mwf_ctx* c, cudaStream_t s);
int read_err_word(mwf_ctx* c, cudaStream_t s, unsigned int* out);
void drop_lists(mwf_ctx* c);
bool use_scan_refresh();

// Host-side work plan of one set of lists (plan.cu): per-group list offsets (padded to tiles), work items, the
// schedules, and the per-group prefix sums the dispatcher needs.
struct Plan {
    std::vector<int64_t> list_off, item_off, inter, split;
    std::vector<WorkItem> items;
};
int plan_cut(mwf_ctx* c, int64_t n_group, const int32_t* grp_first, const int32_t* grp_n, Plan& pl);
int plan_finish(mwf_ctx* c, int64_t n_group, const int32_t* grp_n, const int32_t* n_epj_of, const int32_t* n_spj_of, Plan& pl);
int make_plan(mwf_ctx* c, int64_t n_group, const int32_t* grp_first, const int32_t* grp_n, const int32_t* n_epj_of, const int32_t* n_spj_of, Plan& pl);
void adopt_plan(mwf_ctx* c, Plan& pl, int64_t n_group, const int32_t* grp_first, const int32_t* grp_n, int mode);
int ensure_split_order(mwf_ctx* c, cudaStream_t s);
int ensure_class_order(mwf_ctx* c, cudaStream_t s);
// order_full of the items now on the device (behind their upload on the stream); no host synchronisation
int schedule_full(mwf_ctx* c, int64_t n_items, cudaStream_t s);

// dispatch plumbing shared by the gravity and the short-range dispatches (api_step.cu)
int pick_order(mwf_ctx* c, int64_t g_begin, int64_t g_end, cudaStream_t s, const int32_t** order);
void book_dispatch(mwf_ctx* c, int32_t tag, int64_t g_begin, int64_t g_end);

}  // namespace mwf
