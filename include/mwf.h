/* mwf.h -- C ABI of the B200-native index-based multi-walk force library (libmwf.so).
 *
 * The hot path of "Accelerated FDPS" (arXiv 1907.02290; "P:n" = line n of the paper text the build was
 * written from, SURVEY.md section 8 is the scope contract):
 *
 *   (1) upload / update particles        P:107, P:181, P:391, P:466-474  "send all EPJ and SPJ once"
 *   (2) upload tree cells + index lists  P:181, P:391, P:441-477, P:528-546  lists are INDICES, kept on the device
 *   (3) refresh the monopoles            P:134-136, P:160  moments recomputed every step, also on reuse steps
 *   (4) dispatch the force kernel        P:89 multiwalk, "dispatch", P:557-569 ForceKernelIndex
 *   (5) retrieve acc and pot             P:189 "retrieve", P:595-663 RetrieveKernel
 *   list reuse                           P:115-143, P:242 MAKE_LIST / MAKE_LIST_FOR_REUSE / REUSE_LIST
 *   device-resident reuse step           P:1171-1185 section 7.3 "implement all procedures on the accelerator"
 *
 * Conventions common to every call
 *   - Return value: 0 (MWF_OK) on success, a negative MWF_E* code otherwise (the paper's callbacks return 0,
 *     P:352).  No exceptions, no abort, no exit.  mwf_strerror() gives a text;
 *     mwf_last_cuda_error() the CUDA text behind the last MWF_ECUDA.
 *   - "host" pointers are ordinary CPU memory (pinned memory makes the copies truly asynchronous);
 *     "device" pointers are CUDA global memory on the ctx's device.  Each argument says which.
 *   - Ownership: the caller owns every array it passes.  The library copies what it needs during the
 *     call or on the given stream; host sources of asynchronous copies must stay valid until that stream
 *     has been synchronised (mwf_retrieve() / mwf_sync() do).  All device storage of the library lives in
 *     one arena: either caller-allocated (e.g. a torch tensor) and handed to mwf_create(), or allocated
 *     by the library when arena == NULL.
 *   - Streams are `cudaStream_t` handles passed as `void*` (NULL = the legacy default stream).
 *     Cross-stream ordering (store updates -> refresh -> force kernels -> next store update) is enforced
 *     inside the library with CUDA events; the caller never needs to synchronise between calls.
 *   - Not thread-safe per ctx; distinct ctxs are independent.
 *   - All particle-indexed arrays are in TREE (Morton) ORDER: particle p of group g is
 *     grp_first[g] <= p < grp_first[g] + grp_n[g]; the i-particles ARE the stored j-particles (the
 *     paper's own section 7.3 proposal), so there is no separate EPI upload.
 */
#ifndef MWF_H
#define MWF_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mwf_ctx mwf_ctx; /* opaque */

/* EPJ / SPJ on the device: float4 (x, y, z, m), 16 B.  SPJ = monopole of a tree cell:
 * centre of mass and total mass, same type and same array as EPJ. */
typedef struct { float x, y, z, m; } mwf_posm;
/* FORCE on the device: float4 (ax, ay, az, pot), 16 B. */
typedef struct { float ax, ay, az, pot; } mwf_accp;
/* Velocity on the device: float4 (vx, vy, vz, unused), 16 B so that it moves with vector loads. */
typedef struct { float vx, vy, vz, pad; } mwf_vel;
/* Tree cell: particle range [first_ptcl, first_ptcl + n_ptcl) in tree order and child range
 * [first_child, first_child + n_child) in the cell array (n_child == 0: leaf).  Cell 0 is the root and
 * covers [0, N).  Children of a cell are stored contiguously, after their parent (level order),
 * and their particle ranges partition the parent's range. */
typedef struct { int32_t first_ptcl, n_ptcl, first_child, n_child; } mwf_cell;

typedef struct {
    float eps;          /* Plummer softening length, > 0 (eps^2 must be a normal float)      */
    float G;            /* gravitational constant, applied to acc and pot                    */
    int64_t max_ptcl;   /* capacity: particles                                               */
    int64_t max_cell;   /* capacity: tree cells                                              */
    int64_t max_group;  /* capacity: i-groups                                                */
    int64_t max_entry;  /* capacity: total list entries, EPJ + SPJ summed over groups        */
    int32_t n_tag;      /* number of dispatch tags (= internal streams), 1 .. MWF_MAX_TAG; paper uses 8 */
    int32_t device;     /* CUDA device ordinal                                               */
} mwf_params;

#define MWF_MAX_TAG 16

/* INTERACTION_LIST_MODE of the paper. */
enum { MWF_MAKE_LIST = 0, MWF_MAKE_LIST_FOR_REUSE = 1, MWF_REUSE_LIST = 2 };

enum {
    MWF_OK = 0,
    MWF_EINVAL = -1,  /* null pointer, negative size, eps <= 0, bad tag or mode                          */
    MWF_ESTATE = -2,  /* call out of order: dispatch without lists / with stale monopoles, REUSE_LIST with
                         no saved lists (MAKE_LIST does not keep them), retrieve of an idle tag   */
    MWF_ERANGE = -3,  /* an index, range or offset in the uploaded tree / lists is out of bounds or not
                         monotone (found by the one-time device validation)                               */
    MWF_ENOMEM = -4,  /* exceeds a max_* capacity or the arena is too small                              */
    MWF_ECUDA = -5    /* a CUDA call failed; sticky text via mwf_last_cuda_error()                       */
};

/* Bytes of device memory a ctx with these capacities needs (write to *bytes). */
int mwf_arena_bytes(const mwf_params* p, int64_t* bytes);

/* Create a ctx.  arena: DEVICE pointer to at least mwf_arena_bytes() bytes, 256-B aligned, owned by the
 * caller and kept alive until mwf_destroy(); or NULL to let the library cudaMalloc it. */
int mwf_create(mwf_ctx** out, const mwf_params* p, void* arena, int64_t arena_bytes);
int mwf_destroy(mwf_ctx* c);

/* Bind the caller's stream (e.g. a torch.cuda.Stream) to a tag instead of the internal one. */
int mwf_set_tag_stream(mwf_ctx* c, int32_t tag, void* cuda_stream);

/* (1) Upload or update particles [first, first + n) of the store, tree order (P:466-474 H2dJptcl).
 * src: n records, HOST if src_on_device == 0 else DEVICE.  Asynchronous on `stream`.  Marks the
 * monopoles stale: mwf_refresh_monopoles() must follow before the next dispatch. */
int mwf_set_particles(mwf_ctx* c, const mwf_posm* src, int64_t first, int64_t n, int src_on_device, void* stream);

/* Read back particles [first, first + n) of the store (test / integration hook). dst HOST or DEVICE. Blocking.
 * MWF_ERANGE when the range reaches behind the particles (N once a tree is set, else what has been uploaded). */
int mwf_get_particles(mwf_ctx* c, mwf_posm* dst, int64_t first, int64_t n, int dst_on_device);

/* (2a) Upload the tree topology (construction step only).  cells: n_cell records, HOST.
 * Defines N = cells[0].n_ptcl.  Validated on the device (MWF_ERANGE): particle and child ranges in bounds, children
 * partition their parent, every cell but the root is the child of exactly one cell.  Blocking. */
int mwf_set_tree(mwf_ctx* c, const mwf_cell* cells, int64_t n_cell, void* stream);

/* (2b) Upload the i-groups and their interaction lists as two CSR index lists (construction step only;
 * EPJ indices then SPJ indices: kept on the device).  All arrays HOST.
 *   grp_first[g], grp_n[g]   i-range of group g (any n_i >= 1); groups must be disjoint
 *   epj_off[n_group + 1], epj_id[]   particle indices in [0, N)
 *   spj_off[n_group + 1], spj_id[]   cell indices in [0, n_cell)
 * A group's EPJ list must contain either all of the group's own particles (what a Barnes walk yields;
 * their self terms are excluded) or none of them; anything else is MWF_EINVAL.
 * mode: MWF_MAKE_LIST (lists valid for one evaluation, dropped once every dispatched tag has been
 * retrieved) or MWF_MAKE_LIST_FOR_REUSE (kept until the next mwf_set_lists / mwf_set_tree).
 * Requires mwf_set_tree() first.  Validates on the device, re-encodes into one padded merged list per
 * group and builds the work schedule.  Blocking.
 * Call order and accuracy (reading S11b of DESIGN.md): every SPJ entry is marked here, once, as FAR (swept from its
 * fp32 record) or NEAR (swept with the fp64 remainder of its centre of mass, about 3 x the cost), from the particle
 * positions in the store.  Only positions uploaded for this step are used: all N particles, in the new tree's order,
 * uploaded since the last dispatch (mwf_set_particles from 0 upwards or mwf_swap_store; mwf_build leaves them so).
 * If they arrive only after this call, every SPJ entry is treated as NEAR -- always accurate, slower.  The marks are
 * kept over the reuse steps while the particles drift; FAR allows a margin of 16x over what the error bound needs, so
 * a group and a cell would have to close a sizeable part of their distance before a mark is wrong -- rebuild the lists
 * before that, as the opening criterion needs anyway.  The marks hold for ANY list, also one that no opening
 * criterion produced: the distance used is a lower bound (tight boxes of the group's and of the cell's particles). */
int mwf_set_lists(mwf_ctx* c, int64_t n_group, const int32_t* grp_first, const int32_t* grp_n,
                  const int64_t* epj_off, const int32_t* epj_id, const int64_t* spj_off, const int32_t* spj_id,
                  int mode, void* stream);

/* Declare the kind of step that follows.  MWF_REUSE_LIST: MWF_ESTATE unless lists saved with
 * MWF_MAKE_LIST_FOR_REUSE are present.  MWF_MAKE_LIST*: drops any saved lists; mwf_set_tree() and
 * mwf_set_lists() must follow. */
int mwf_begin_step(mwf_ctx* c, int mode);

/* (3) Recompute the monopole (total mass, centre of mass) of every tree cell from the current particle
 * store, bottom-up over the fixed tree, on the device, and write them as SPJ entries behind the
 * particles.  Asynchronous on `stream`. */
int mwf_refresh_monopoles(mwf_ctx* c, void* stream);

/* (4) Launch the force kernel over groups [g_begin, g_end) on the stream of `tag`; non-blocking.
 * For every particle i of those groups, over the group's list (reading S1-S5 of DESIGN.md):
 *   acc_i =  G sum_k m_k (x_k - x_i) / (|x_k - x_i|^2 + eps^2)^(3/2)
 *   pot_i = -G sum_k m_k / (|x_k - x_i|^2 + eps^2)^(1/2)        (k != i by index)
 * First-call latency: a dispatch over all groups, or over one of the ranges of mwf_get_tag_split(), uses a schedule made
 * with the lists.  The FIRST dispatch over any other range after new lists builds, on the host, the permutation that
 * orders the work items of arbitrary ranges widest first (about 1 ms for 10^5 items, plus one upload); later ones reuse it.
 * MWF_ECUDA when no block of the kernel fits an SM (never a silent empty launch). */
int mwf_dispatch(mwf_ctx* c, int32_t tag, int64_t g_begin, int64_t g_end);

/* ---- Method G1 of the paper, for A/B comparison with the index method (paper
 * P:170-177 "multiwalk", Fig. 2 DispatchKernelStream, Table 1, Fig. 5): the interaction list of every
 * group carries the j-particle DATA (16 B per entry) instead of 4-byte indices, and is sent with every
 * dispatch -- on reuse steps too, because particle data changes every step.
 *
 * mwf_reserve_data_lists: allocate (cudaMalloc, outside the arena) one staging buffer of max_entry_per_tag j
 * records per tag; frees any earlier reservation.  MWF_ESTATE while a tag is in flight.
 * mwf_dispatch_data: like mwf_dispatch over groups [g_begin, g_end), but group g_begin + k interacts with the
 * records jdata[joff[k] .. joff[k+1]) (EPJ records, then the SPJ records = monopoles of its list's cells) instead
 * of gathering through its index list.  jdata: HOST (pinned for overlap) or DEVICE, joff: HOST, ng + 1 offsets in
 * records, joff[0] == 0; both are copied on the tag's stream, so they must stay valid until the tag is retrieved.
 * The groups, their i-ranges, the self-exclusion rule and the work schedule are those of the lists given to
 * mwf_set_lists()/mwf_build(); each run must have exactly the length of the group's index list (MWF_ERANGE).
 * The i-particles are read from the store; the monopoles need not be fresh (SPJ data travels in jdata).
 * MWF_ENOMEM when joff[ng] exceeds the reservation, MWF_ESTATE when the tag has not been retrieved yet. */
int mwf_reserve_data_lists(mwf_ctx* c, int64_t max_entry_per_tag);
int mwf_dispatch_data(mwf_ctx* c, int32_t tag, int64_t g_begin, int64_t g_end, const mwf_posm* jdata, const int64_t* joff,
                      int jdata_on_device);

/* ---- Quadrupole SPJ (the paper computes "multipole moments" of the cells, and
 * measures the monopole case).  order = 1 (default): an SPJ entry is a point mass at the cell's centre of mass.
 * order = 2: it also carries Q = sum m (x - X)(x - X)^T about the centre of mass X and acts through the second-order
 * Taylor expansion of the same softened kernel (reading S22 of DESIGN.md; R = X - x_i, s^2 = |R|^2 + eps^2):
 *     pot_i -= G [ M/s - tr(Q)/(2 s^3) + 3 (R.Q.R)/(2 s^5) ]
 *     acc_i += G [ M R/s^3 - 3 tr(Q) R/(2 s^5) - 3 (Q R)/s^5 + 15 (R.Q.R) R/(2 s^7) ]
 * mwf_refresh_monopoles() then also computes Q bottom-up (parallel-axis theorem, fp64), and every mwf_dispatch()
 * runs the order-2 force kernel: the same sweep over the same lists, with the Q terms of the SPJ entries evaluated
 * from the same distances and reciprocal square roots as their monopole terms (one kernel, one pass over the lists).
 * Allocates 80 B per max_cell with cudaMalloc on first use (MWF_ENOMEM); marks the moments stale when the order
 * changes; MWF_ESTATE while a tag is in flight or unretrieved.  mwf_dispatch_data() supports order 1 only. */
int mwf_set_spj_order(mwf_ctx* c, int order);
/* Test hook: 8 floats per cell (Qxx Qyy Qzz Qxy Qxz Qyz tr(Q)/2 0) as the refresh stored them.  dst HOST or DEVICE. */
int mwf_get_quadrupoles(mwf_ctx* c, float* dst, int dst_on_device);

/* ---- Short-range workload through the same index lists (paper P:79: "In the case of
 * short-range interaction such as SPH interaction between particles, we still use treewalk but with cell-opening
 * criterion different from the standard opening angle"; particle records "much larger in the case of SPH";
 * such lists can be reused because the time step is stability-limited).  The lists are EPJ-only neighbour
 * lists given to mwf_set_lists() (all spj offsets 0): every particle k with |x_i - x_k| < 2 max(h_i, h_k) for some i
 * of the group must be in the group's list; extra entries cost time, never accuracy (compact support).  The paper
 * prints no SPH formula; reading S23 of DESIGN.md takes the cubic-spline (M4) kernel with support 2h,
 *     W(r,h) = 1/(pi h^3) { 1 - 3/2 q^2 + 3/4 q^3 (q < 1); 1/4 (2 - q)^3 (1 <= q < 2); 0 (q >= 2) },  q = r/h.
 * Per-particle record, tree order, 16 B: smoothing length h > 0, specific internal energy u, density rho,
 * P/rho^2.  mwf_set_sph() uploads records [first, first + n) (all four fields; HOST or DEVICE source, asynchronous on
 * `stream`; the array is cudaMalloc'ed on first use, 16 B x max_ptcl, MWF_ENOMEM); mwf_get_sph() reads them back
 * (blocking).
 *
 * mwf_dispatch_density: for every particle i of groups [g_begin, g_end), on the stream of `tag`, non-blocking:
 *     rho_i = sum_{k in list} m_k W(|x_i - x_k|, h_i)      (gather form, self term included)
 *     (P/rho^2)_i = (gamma - 1) u_i / rho_i                (ideal gas; gamma > 1 else MWF_EINVAL)
 *   written into the rho and P/rho^2 fields of the records.  mwf_retrieve(tag, dst, ..) then copies the RECORDS of those
 *   particles (dst is an array of mwf_sph indexed by tree position); dst == NULL just waits.
 * mwf_dispatch_hydro: pressure-gradient acceleration with the symmetrised kernel gradient,
 *     a_i = - sum_{k != i} m_k [(P/rho^2)_i + (P/rho^2)_k] 1/2 [gradW(r_ik, h_i) + gradW(r_ik, h_k)],
 *   gradW(r, h) = dW/dr (x_i - x_k)/r (a pair at zero distance contributes nothing), written as (ax, ay, az, 0) into
 *   the result array that mwf_retrieve() copies out.  Reads h and P/rho^2 of every listed particle: these must be
 *   current (from density dispatches over all groups, or uploaded); the library orders a hydro dispatch behind the
 *   density kernels in flight on every tag.
 * Both need the tree, the lists, particles and records for all N (MWF_ESTATE otherwise); no monopoles are involved,
 * and lists that hold SPJ entries (gravity lists) are refused with MWF_ESTATE.
 * A tag holds one kind of result at a time: MWF_ESTATE when its previous results of the other kind (records vs
 * accelerations) have not been retrieved.  Lists set with MWF_MAKE_LIST stay until the next mwf_begin_step /
 * mwf_set_lists (a step needs them twice).  Artificial viscosity and the energy equation are not evaluated. */
typedef struct { float h, u, rho, pr2; } mwf_sph;
int mwf_set_sph(mwf_ctx* c, const mwf_sph* src, int64_t first, int64_t n, int src_on_device, void* stream);
int mwf_get_sph(mwf_ctx* c, mwf_sph* dst, int64_t first, int64_t n, int dst_on_device);
int mwf_dispatch_density(mwf_ctx* c, int32_t tag, int64_t g_begin, int64_t g_end, float gamma);
int mwf_dispatch_hydro(mwf_ctx* c, int32_t tag, int64_t g_begin, int64_t g_end);
/* One whole short-range evaluation for a step whose tree and neighbour lists are already on the device (the analogue of
 * mwf_calc_force_all): upload all N particles (src HOST or DEVICE; NULL = keep the store) and all N records (rec: h and
 * u are read), density pass over all groups, records back into rec (rho and P/rho^2 filled in), hydro pass over all
 * groups, accelerations into dst.  With a host rec or dst the groups are split over the tags so that every tag's copy
 * overlaps the other tags' kernels.  Blocking. */
int mwf_calc_sph_all(mwf_ctx* c, const mwf_posm* src, int src_on_device, mwf_sph* rec, int rec_on_device, mwf_accp* dst, int dst_on_device,
                     float gamma);

/* (5) Copy acc+pot of the particles of every group dispatched under `tag` since its last retrieve into
 * dst and wait for it.  dst: base of an N-record array indexed by tree-order particle
 * position, HOST or DEVICE; records of other particles are not touched.  dst == NULL: wait for the tag and
 * discard its results (they stay in the library's result array; a device-resident loop needs no copy). */
int mwf_retrieve(mwf_ctx* c, int32_t tag, mwf_accp* dst, int dst_on_device);

/* One whole evaluation, the analogue of calcForceAllAndWriteBackMultiWalkIndex for a step
 * whose tree and lists are already on the device: upload all N particles (src HOST or DEVICE; NULL = keep
 * the store), refresh, dispatch all groups split over the tags, retrieve everything into dst. */
int mwf_calc_force_all(mwf_ctx* c, const mwf_posm* src, int src_on_device, mwf_accp* dst, int dst_on_device);

/* ---- Pipelined host loop ("all of these can be overlapped", P:189 dispatch / retrieve split): the particles of the
 * NEXT step are written into a second (shadow) store while the force kernels of the current step still read the current
 * one, so that a host that integrates tag by tag hides the H2D copy of eq. 18's first term under the kernels:
 *     for every tag t in dispatch order:  mwf_retrieve(t, dst)            results of step k of that tag's particles (D2H)
 *                                         (the host integrates them)
 *                                         mwf_set_particles_next(...)     their positions of step k+1 (H2D, own stream)
 *     mwf_swap_store(); mwf_refresh_monopoles(); mwf_dispatch(t, ...) for every tag      step k+1
 * mwf_set_particles_next: like mwf_set_particles, into the shadow store; asynchronous on `stream`, waits for nothing
 *   (no kernel reads the shadow store); needs a tree (MWF_ESTATE), [first, first + n) inside [0, N) (MWF_ERANGE).
 * mwf_swap_store: the shadow store becomes the store.  MWF_ESTATE unless the ranges written since the last swap tile
 *   [0, N) exactly (no hole, no overlap) and no tag is in flight (every dispatched tag retrieved).  Everything
 *   enqueued later on any stream through this library is ordered behind the shadow uploads.  The monopoles become
 *   stale (mwf_refresh_monopoles must follow); velocities, results, tree and lists are not touched.
 * mwf_get_tag_split: bounds[0 .. n_tag] = the group ranges [bounds[t], bounds[t+1]) that mwf_calc_force_all dispatches
 *   per tag (MWF_ESTATE without lists): by interaction count, equal shares for the first half of the tags, then shares
 *   falling linearly to an eighth for the last tag -- the tags finish in order, the copies of a tag hide behind the
 *   kernels of the tags after it, and the copies of the last tag, which nothing hides, are small. */
int mwf_set_particles_next(mwf_ctx* c, const mwf_posm* src, int64_t first, int64_t n, int src_on_device, void* stream);
int mwf_swap_store(mwf_ctx* c, void* stream);
int mwf_get_tag_split(mwf_ctx* c, int64_t* bounds);

/* ---- Device-side construction step (paper P:149-172: root cell, Morton keys,
 * radix sort, reorder, cells linked level by level, one tree walk per i-group emitting an index list).  Works on
 * the particles [0, n) currently in the store, in ANY order: sorts them (and the velocities, when all n have been
 * uploaded) into tree order in place, builds cells, groups and lists on the device and leaves the ctx in the
 * state mwf_set_tree() + mwf_set_lists(mode) leave it in.  Readings O1-O4 of DESIGN.md (the same as the host
 * builder's): cube root cell padded by 2^-10, 21 key bits per axis, leaf = at most n_leaf particles, group =
 * first cell on a root path with at most n_grp particles, open iff cell side > theta x distance from the cell
 * centre to the group's particle bounding box.  theta in [0, 1].  Results of the previous step must have been
 * retrieved (MWF_ESTATE otherwise).  MWF_ENOMEM when max_cell / max_group / max_entry are too small; the particles
 * (velocities, SPH records) have then already been sorted in place, so they count as not uploaded any more: upload them
 * again before the next attempt.  Blocking (stream synchronisations to size the tree levels, after the counting walk and
 * at the end; the host cuts and schedules the work items while the device walks the tree). */
int mwf_build(mwf_ctx* c, int64_t n, int32_t n_leaf, int32_t n_grp, double theta, int mode, void* stream);
/* The same construction step for the short-range workload (NEXT-4): the list walk uses the neighbour-search criterion
 * of reading S24 instead of the opening angle -- a cell is opened iff the gap between its cube and the group's particle
 * box is <= max(R_g, R_c), R = 2 (1 + skin) x the largest smoothing length among the group's / the cell's particles;
 * opened leaves give EPJ entries, nothing else is listed (no SPJ).  Needs the SPH records of particles [0, n)
 * (mwf_set_sph, in the same order as the particles; MWF_ESTATE otherwise); they are sorted into tree order with the
 * particles (mwf_build does the same when all n records have been uploaded).  skin >= 0. */
int mwf_build_neighbours(mwf_ctx* c, int64_t n, int32_t n_leaf, int32_t n_grp, double skin, int mode, void* stream);
/* Sizes of what mwf_build() / mwf_build_neighbours() made. */
int mwf_get_build_sizes(mwf_ctx* c, int64_t* n_cell, int64_t* n_group, int64_t* n_epj, int64_t* n_spj, int32_t* n_level);
/* perm[p] = index, in the order the particles were uploaded, of the particle now at tree position p. */
int mwf_get_permutation(mwf_ctx* c, int32_t* perm, int dst_on_device);
/* Read-back hooks (HOST destinations): cells (n_cell records) and their geometry (centre x,y,z and side, fp64;
 * only for a device-built tree); group ranges; the lists in the CSR form mwf_set_lists() takes. */
int mwf_get_tree(mwf_ctx* c, mwf_cell* cells, double* geom4);
int mwf_get_groups(mwf_ctx* c, int32_t* grp_first, int32_t* grp_n);
int mwf_get_lists(mwf_ctx* c, int64_t* epj_off, int32_t* epj_id, int64_t* spj_off, int32_t* spj_id);
/* The list buffers exactly as the force kernel reads them (pin P9 of SURVEY.md 8(c): "list buffers bit-identical before /
 * after the reuse steps"): list_off[n_group + 1] (offsets in entries, multiples of 64) and the merged,
 * padded index list (per group: run 1 = EPJ ids then FAR SPJ ids + N, dummy indices up to a whole tile; run 2 = NEAR SPJ ids + N, dummy indices up to a whole tile).  *n_group, *n_entry = groups and
 * entries in the merged list (also without destinations: call once to size them).  Destinations HOST or DEVICE, either may be NULL.
 * MWF_ESTATE without lists.  Blocking. */
int mwf_get_list_buffer(mwf_ctx* c, int64_t* list_off, int32_t* list, int64_t* n_group, int64_t* n_entry, int dst_on_device);
/* The third array the force kernel reads with them: run1_len[g] = entries of group g's run 1 (its EPJ entries + its FAR SPJ
 * entries, reading S11b); run 2 (the NEAR SPJ entries) starts at the next multiple of 64 behind it.  n_group values, HOST or
 * DEVICE.  MWF_ESTATE without lists.  Blocking. */
int mwf_get_run1_len(mwf_ctx* c, int32_t* run1_len, int dst_on_device);

/* ---- Device-resident reuse step (the paper's own conclusion, P:1171-1185:
 * with the lists resident the per-step host<->device transfers of particles and forces are what is left,
 * so the orbit integration (the paper's step 5) moves to the device as well).  Kick-drift-kick
 * leapfrog in fp32 on the store (reading S14b of DESIGN.md):
 *     mwf_kick_drift:  v += acc * dt/2 ;  x += v * dt        (marks the monopoles stale)
 *     mwf_kick:        v += acc * dt/2
 * acc is the result array of the last evaluation, read in place; both calls return MWF_ESTATE unless
 * every group has been dispatched since the positions last changed and velocities for all N particles
 * have been uploaded.  Asynchronous on `stream`; ordered after the force kernels by the library. */

/* Upload / read back velocities [first, first + n), tree order.  src/dst HOST or DEVICE. */
int mwf_set_velocities(mwf_ctx* c, const mwf_vel* src, int64_t first, int64_t n, int src_on_device, void* stream);
int mwf_get_velocities(mwf_ctx* c, mwf_vel* dst, int64_t first, int64_t n, int dst_on_device);
int mwf_kick_drift(mwf_ctx* c, float dt, void* stream);
int mwf_kick(mwf_ctx* c, float dt, void* stream);
/* One whole list-reuse step with no host transfer, all on the stream of tag 0 and non-blocking:
 * begin_step(MWF_REUSE_LIST), kick_drift(dt), refresh_monopoles, dispatch of all groups, kick(dt).
 * mwf_retrieve(c, 0, ...) afterwards copies out acc+pot of all particles; mwf_sync() just waits. */
int mwf_step_reuse(mwf_ctx* c, float dt);

/* Test hooks: monopoles as stored (float4 per cell) and device-side results without a copy. */
int mwf_get_monopoles(mwf_ctx* c, mwf_posm* dst, int dst_on_device);
/* DEVICE pointers into the arena: store (N particles then n_cell SPJ) and result array. */
int mwf_device_pointers(mwf_ctx* c, mwf_posm** store, mwf_accp** accp);

/* ---- The monopole pass for callers that must not allocate device memory.
 * Everything above works through an mwf_ctx, whose arena somebody has to allocate.  Some callers cannot: a plugin inside
 * an application whose own pool owns the GPU's memory (a guest cudaMalloc may be refused or against the rules), a routine
 * on a latency-bound path (cudaMalloc and cudaFree synchronise the whole device), code on a nearly full GPU where the
 * allocation is the one call that may fail.  mwf_monopoles_static() needs no ctx and allocates nothing, on the host side
 * of CUDA or the device side: its working memory (fp64 moments, parent links, arrival counters; 40 B per cell) is one
 * fixed array inside the library image, sized for MWF_STATIC_MAX_CELL cells (5 MiB).  Every GPU that loads the library
 * holds that array until the process exits, which is why the limit is modest; larger trees need an mwf_ctx.
 *
 * Computes, for every cell c of the tree, the record (centre of mass x, y, z, total mass) of the particles in its range,
 * summed in fp64 bottom-up (leaf sums, then children in child order) and rounded once to float -- the
 * records mwf_refresh_monopoles() + mwf_get_monopoles() give for the same tree and particles, to the last float bit or
 * one (the ctx path sums by a prefix scan).  A cell of zero mass gets its first particle's position and mass 0.
 *   cells   DEVICE, n_cell records laid out as mwf_set_tree() wants them (children behind their parent, child ranges
 *           partitioning the parent's).  NOT validated (that needs a read-back): ranges that leave the arrays are
 *           clipped or ignored, so a malformed tree gives wrong records, never an out-of-bounds access.
 *   ptcl    DEVICE, n_ptcl records in tree order.       spj   DEVICE, n_cell records, written.
 *   All three 16-byte aligned, on the CURRENT device (there is no ctx to name one), owned by the caller and valid until
 *   the work on `stream` has finished.  Asynchronous on `stream`; the caller synchronises.
 * Returns MWF_ENOMEM when n_cell > MWF_STATIC_MAX_CELL, MWF_EINVAL for null / misaligned pointers or sizes <= 0,
 * MWF_ECUDA when a CUDA call fails; mwf_static_last_error() gives this thread's last message in words.
 * First call on a device: it also looks up the array's device address (once per device).  Make that call before any
 * stream capture begins.
 * Sharing: all calls on a GPU use the same array, which keeps the previous call's contents; each call resets, on its
 * stream, what it needs clean.  Calls that overlap on one GPU (two streams, two threads) race on it -- run them one
 * after the other. */
#define MWF_STATIC_MAX_CELL 131072
int mwf_monopoles_static(const mwf_cell* cells, int64_t n_cell, const mwf_posm* ptcl, int64_t n_ptcl, mwf_posm* spj, void* stream);
const char* mwf_static_last_error(void);

/* Wait for everything the ctx has enqueued. */
int mwf_sync(mwf_ctx* c);

/* Counters since creation: kernels launched by the library, interactions dispatched (sum n_i * n_list,
 * padding excluded), entries resident in the merged list (padding included). */
int mwf_get_counters(mwf_ctx* c, int64_t* kernel_launches, int64_t* interactions, int64_t* padded_entries);

/* Timing hook: CUDA-event time in ms of the force kernels of the last mwf_dispatch on `tag`
 * (valid after that tag's stream was synchronised). */
int mwf_last_dispatch_ms(mwf_ctx* c, int32_t tag, float* ms);

const char* mwf_strerror(int code);
const char* mwf_last_cuda_error(mwf_ctx* c);

#ifdef __cplusplus
}
#endif
#endif /* MWF_H */
