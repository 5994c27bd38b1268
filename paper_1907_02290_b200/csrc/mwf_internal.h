// Internal declarations shared by the translation units of libmwf.so (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "mwf.h"

namespace mwf {

constexpr int TILE_J = 64;          // j entries staged per warp tile; merged lists are padded to this
#ifndef MWF_WARPS_PER_CTA
#define MWF_WARPS_PER_CTA 8
#endif
constexpr int WARPS_PER_CTA = MWF_WARPS_PER_CTA;    // force kernel block
constexpr int SMALL_CTA_WARPS = 2;  // block of a sub-wave dispatch (one item per warp)
constexpr int SCHED_WINDOWS = 16;    // Morton windows of the work schedule when the store exceeds the L2
constexpr int CHUNK_I = 64;         // i-particles of a full work item (2 per lane)
constexpr int MIN_WIDTH = 2;        // narrowest item: 2 lanes x 2 i-particles, 16 j-slices
constexpr int N_WIDTH_CLASS = 5;    // widths 32, 16, 8, 4, 2
inline int width_class(int width) { return width >= 32 ? 0 : width >= 16 ? 1 : width >= 8 ? 2 : width >= 4 ? 3 : 4; }
// An SPJ entry is FAR when the cell's coordinates are at most this many times its distance from the group: the fp32
// rounding of its centre of mass, at most 2^-24 of the coordinate, is then within 32 * 2^-24 = 1.9e-6 of the separation, i.e.
// at most 6e-6 of that entry's term and of the order of the kernel's other rounding errors (the north_star bound is 1e-4 on
// the whole acceleration; measured maxima per config: profiles/r02_acceptance.md), and the entry is swept like a particle,
// from its 16-byte record in the caller's coordinates.  NEAR entries are swept in item-centred coordinates with the
// rounding remainder (reading S11b).  kappa = 4 costs 3.5 % on config 5 (31 % of the SPJ entries near instead of none).
#ifndef MWF_KAPPA
#define MWF_KAPPA 32.f
#endif
constexpr float SPJ_FAR_KAPPA = MWF_KAPPA;

// One unit of work for one warp: n_i <= 2 * width consecutive i-particles of one group against the
// group's whole list.  width = 32, 16, 8, 4 or 2 lanes hold the i-particles (2 per lane); the warp is
// split into 32 / width slices that share them and take every (32 / width)-th j-pair.
struct WorkItem {
    int32_t i_first;
    int32_t n_i;
    int32_t group;
    int32_t width;
};

// Modelled cost of an item per list tile, in issue cycles of its warp: staging + width j-pairs x 2 i.
// Used on the host to cut groups into items and to order the items longest-first.
#ifndef MWF_COST_STAGE
#define MWF_COST_STAGE 40
#endif
// j-pairs of a tile unrolled in the W = 32 / 16 sweeps of run 1: 16, not all 32 -- the kernel then is 79 KB of SASS; beyond
// ~95 KB its time falls off a cliff (instruction fetch of 16 warps in differently specialised loops, profiles/r02_kforce_variants.md)
#ifndef MWF_UNROLL_WIDE
#define MWF_UNROLL_WIDE 16
#endif
#ifndef MWF_FLUSH_MIN
#define MWF_FLUSH_MIN 2
#endif
#ifndef MWF_MIN_CTAS
#define MWF_MIN_CTAS 2
#endif
constexpr int64_t COST_STAGE = MWF_COST_STAGE;
constexpr int64_t COST_PAIR = 33;
inline int64_t item_cost_per_tile(int width) { return COST_STAGE + COST_PAIR * width; }

struct ForceArgs {
    const float4* store;        // particles then SPJ then one zero-mass dummy
    const float4* spj_lo;       // [n_cell + 1] per cell: the rounding remainder of the SPJ record's centre of mass (entry n_cell: zero)
    int32_t n_ptcl;             // list indices >= n_ptcl are SPJ entries
    int32_t dummy;              // index of the zero-mass record (n_ptcl + n_cell)
    const int32_t* run1_len;    // per group: entries of run 1 (EPJ + far SPJ; 16-byte records, caller's coordinates); run 2
                                //   (near SPJ; 32-byte records, item-centred) starts at the next tile boundary
    const int32_t* list;        // merged, padded lists
    const int64_t* list_off;    // per group, in entries (multiples of TILE_J)
    const uint8_t* grp_self;    // 1: the group's own particles are in its EPJ list
    const WorkItem* items;
    const int32_t* order;       // cost-sorted permutation of item indices, or nullptr = identity
    int32_t n_seg;              // > 0: the dispatch is n_seg runs of `order` (the class-sorted permutation), widest items first:
    int64_t seg_begin[N_WIDTH_CLASS];      //   work index w in [seg_cum[k], seg_cum[k + 1]) is order[seg_begin[k] + w - seg_cum[k]]
    int64_t seg_cum[N_WIDTH_CLASS + 1];
    const float4* jdata;        // method G1 (data lists): j records of groups [g_base, ...), else nullptr
    const int64_t* joff;        // G1: offsets of those groups' runs in jdata, in records
    int64_t g_base;
    float4* accp;
    unsigned int* counter;      // dynamic scheduling counter (zeroed before launch), or nullptr = static
    int64_t item_begin;
    int64_t n_items;
    float eps2;
    float G;
    const float4* quad;         // order 2 (NEXT-3): two float4 per cell (Qxx Qyy Qzz Qxy) (Qxz Qyz tr(Q)/2 0), else nullptr
    const int32_t* n_far;       // order 2: per group, the far SPJ entries of run 1 (the EPJ entries are run1_len - n_far)
    int32_t n_cell;
    float4* vel;                // non-null: the closing kick of the leapfrog in the epilogue, v += acc * kick_h (NEXT-1)
    float kick_h;
};

// Short-range workload (NEXT-4, sph_kernel.cu): same lists, items and schedule as the force kernel.
struct SphArgs {
    const float4* store;
    float4* sph;                // per particle (h, u, rho, P/rho^2): density writes the last two, hydro reads h and P/rho^2
    const int32_t* list;
    const int64_t* list_off;
    const WorkItem* items;
    const int32_t* order;
    float4* accp;               // hydro: (ax, ay, az, 0)
    unsigned int* counter;
    int64_t item_begin;
    int64_t n_items;
    int64_t n_ptcl;
    float gamma_m1;             // density: adiabatic index - 1
};
cudaError_t launch_sph(const SphArgs& a, bool hydro, int grid, cudaStream_t s);
int sph_max_ctas_per_sm(bool hydro);

// kernels' host launchers (defined next to their kernels)
cudaError_t launch_force(const ForceArgs& a, int grid, int warps_per_cta, cudaStream_t s);
int force_max_ctas_per_sm();
int force_quad_max_ctas_per_sm();

cudaError_t launch_tree_prepare(const mwf_cell* cells, int64_t n_cell, int64_t max_ptcl, int32_t* parent, int32_t* counter,
                                unsigned int* err, cudaStream_t s);
// quad64 / quad non-null: also the second moments about the centres of mass (6 doubles per cell) and their float record
cudaError_t launch_monopoles(const mwf_cell* cells, const int32_t* parent, int64_t n_cell, int64_t n_ptcl, float4* store, float4* spj_lo,
                             double4* mom64, int32_t* counter, double* quad64, float4* quad, cudaStream_t s);
// scan variant of the refresh (monopole_kernel.cu): leaf ranking at the construction step, then leaf sums + prefix scan per refresh
int64_t scan4_tiles(int64_t n_leaf_cells);
cudaError_t launch_leaf_ranking(const mwf_cell* cells, int64_t n_cell, int64_t n_ptcl, int32_t* mark, int32_t* scratch, int2* cell_lr,
                                int32_t* n_leaf_pinned, cudaStream_t s);
cudaError_t launch_monopoles_scan(const mwf_cell* cells, const int2* cell_lr, int64_t n_cell, int64_t n_ptcl, int64_t n_leaf_cells, float4* store,
                                  float4* spj_lo, double4* P, double4* toff, cudaStream_t s);
cudaError_t launch_classify_spj(int64_t n_group, const int32_t* grp_first, const int32_t* grp_n, const int64_t* spj_off, int32_t* spj_id,
                                const mwf_cell* cells, const int32_t* parent, int32_t* counter, float4* box, const float4* store, int64_t n_ptcl,
                                int64_t n_cell, bool have_ptcl, int32_t* n_far, cudaStream_t s);
cudaError_t launch_merge_lists(int64_t n_group, const int32_t* grp_first, const int32_t* grp_n, const int64_t* epj_off,
                               const int32_t* epj_id, const int64_t* spj_off, const int32_t* spj_id, const int64_t* list_off,
                               const int32_t* n_far, int32_t* run1_len, int64_t n_ptcl, int64_t n_cell, int32_t* list, uint8_t* grp_self,
                               unsigned int* err, cudaStream_t s);

// ---- work schedule on the device (sched_kernel.cu)
struct SchedBuffers {
    int64_t* cost; int64_t* cum;                 // [max_items + 1]
    uint64_t* key_a; uint64_t* key_b;            // [max_items]
    int32_t* idx_a; int32_t* idx_b;              // [max_items]
    int32_t* seg;                                // [2 * max windows + 1]
    int32_t* hist; int32_t* scan_scratch; int64_t* scan_scratch64;  // scratch of the sort and the scans
};
struct SchedTags {                               // one window per tag: bound[t] = first group of tag t (n_tag = 0: not by tag)
    int32_t n_tag;
    int32_t bound[MWF_MAX_TAG + 1];
};
cudaError_t launch_schedule(const SchedBuffers& b, const WorkItem* items, int64_t n_items, const int64_t* list_off, int n_win, const SchedTags& tags,
                            int32_t* order, cudaStream_t s);

// ---- device-side construction step (NEXT-2): buffers carved from the arena, see build_tree.cu / build_lists.cu
constexpr int WALK_STACK = 6144;  // >= 22 levels x 256 cells (bound derived in build_lists.cu)

struct BuildBuffers {
    float4* store; float4* vel; float4* tmp16;          // tmp16 aliases the result array (free during construction)
    uint64_t* key_a; uint64_t* key_b; int32_t* idx_a; int32_t* idx_b;
    int32_t* hist; int32_t* scan_scratch; int64_t* scan_scratch64;
    float* bbox_part; double* root;
    mwf_cell* cells; double4* geom; int32_t* parent; int32_t* level_cnt; int32_t* level_bounds; int64_t level_cap;
    int32_t* mark; int32_t* grp_cell; int32_t* grp_first; int32_t* grp_n; float* grp_box;
    int32_t* n_epj; int32_t* n_spj; int32_t* n_far; int32_t* run1_len; int64_t* list_off; int64_t* epj_off; int64_t* spj_off; int32_t* list;
    int32_t* walk_stacks; unsigned int* walk_counter; unsigned int* err;
    int32_t* h_i32;                                     // pinned host memory, 2 ints: the per-level and group counts on their way back
};

cudaError_t build_tree_device(const BuildBuffers& b, int64_t n, int n_leaf, int n_grp, int64_t max_cell, int64_t max_group, bool with_vel, float4* sph,
                              int64_t* n_cell_out, int64_t* n_group_out, int* n_level_out, cudaStream_t s);
int64_t walk_warps(int64_t max_group);
// Which cells a group's walk opens: the opening angle (gravity) or the short-range neighbour search (reading S24:
// gap between cell cube and group box <= max over (group, cell) of reach x the largest smoothing length).
struct WalkRule {
    double theta = 0.0;
    bool neighbours = false;
    double reach = 0.0;          // 2 (1 + skin)
    const float* cell_h = nullptr;  // [n_cell] largest h among the cell's particles
    const float* grp_h = nullptr;   // [n_group]
};
// totals_pinned[0..2] (pinned host memory) = padded entries, EPJ entries, SPJ entries, valid once the stream has been synchronised
cudaError_t build_lists_count(const BuildBuffers& b, int64_t n_group, const WalkRule& rule, int64_t n_warps, int64_t* totals_pinned, cudaStream_t s);
cudaError_t build_lists_fill(const BuildBuffers& b, int64_t n_group, const WalkRule& rule, int64_t n_warps, int64_t n_ptcl, int64_t n_cell, cudaStream_t s);
// cell_h / grp_h of a WalkRule from the h field of the SPH records (tree order)
cudaError_t build_smoothing_reach(const BuildBuffers& b, const float4* sph, int64_t n_cell, int64_t n_group, float* cell_h, float* grp_h, cudaStream_t s);
cudaError_t unmerge_lists(const BuildBuffers& b, int64_t n_group, int64_t n_ptcl, int32_t* epj_id, int32_t* spj_id, cudaStream_t s);

cudaError_t launch_kick_drift(float4* store, float4* vel, const float4* accp, int64_t n, float dt, cudaStream_t s);
cudaError_t launch_kick(float4* vel, const float4* accp, int64_t n, float dt, cudaStream_t s);

// bits of the device-side validation word
enum : unsigned int {
    ERR_CELL_RANGE = 1u,     // cell particle range outside [0, N) or empty
    ERR_CHILD_RANGE = 2u,    // child range outside (c, n_cell)
    ERR_CHILD_PART = 4u,     // children do not partition the parent's particle range
    ERR_EPJ_INDEX = 8u,      // EPJ index outside [0, N)
    ERR_SPJ_INDEX = 16u,     // SPJ index outside [0, n_cell)
    ERR_SELF_MIXED = 32u,    // a group's EPJ list holds some but not all of its own particles
    ERR_GROUP_RANGE = 64u,   // group i-range outside [0, N)
    ERR_BUILD_CAPACITY = 128u  // device-side construction: more cells than max_cell
};

}  // namespace mwf
