// Host-side input builder for the index-based multi-walk force path: octree, i-groups and
// per-group interaction lists (indices only).  This is HARNESS code ("H"):
// it produces the inputs both the CUDA library and the CPU oracle consume and holds none of the
// method's arithmetic (no monopoles, no forces) -- the opening test is purely geometric.
//
// Follows the paper's construction step:
//   P:149      root cell from the positions of all particles
//   P:153-156  local tree: Morton keys -> sort -> reorder -> link cells level by level, top to bottom
//   P:77, P:87 Barnes' vectorisation: one tree walk per *group* of particles, one shared list
//   P:181      index method: the list holds indices of EPJ (particles) and SPJ (tree cells)
//   P:401      parameters: theta, max particles per leaf (n_leaf), max particles per group (n_grp)
// Readings where the paper is silent (S6-S9): cube root cell padded by 2^-10,
// 21 bits per axis, geometric-centre-to-group-box distance, open iff l > theta * d.
//
// Plain C ABI so Python can drive it through ctypes.  Compile with -ffp-contract=off: the geometry
// must round exactly like the plain Python restatement the tests compare against.
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#include <parallel/algorithm>
#endif

namespace {

constexpr int KEY_BITS = 21;  // per axis -> 63-bit keys (paper: 64-bit keys)

struct Cell {
    int32_t first_ptcl, n_ptcl, first_child, n_child;
};

struct Tree {
    int64_t n = 0;
    int n_leaf = 0, n_grp = 0;
    double root_c[3] = {0, 0, 0}, root_side = 0;
    std::vector<uint64_t> key;    // sorted
    std::vector<int32_t> perm;    // sorted position -> original index
    std::vector<double> pos;      // sorted, 3 per particle (fp32 values widened)
    std::vector<Cell> cell;       // level (BFS) order
    std::vector<double> geom;     // per cell: centre x,y,z, side
    std::vector<int32_t> level;   // per cell
    std::vector<int32_t> level_first;  // n_level + 1
    std::vector<int32_t> grp_cell, grp_first, grp_n;
    // list blocks (filled by bh_build_lists, drained by bh_get_lists)
    std::vector<std::vector<int32_t>> blk_epj, blk_spj;
    std::vector<int64_t> epj_off, spj_off;
    int64_t blk_groups = 0;
};

inline uint64_t spread3(uint64_t v) {  // 21 bits -> every third bit
    v &= 0x1fffffULL;
    v = (v | v << 32) & 0x1f00000000ffffULL;
    v = (v | v << 16) & 0x1f0000ff0000ffULL;
    v = (v | v << 8) & 0x100f00f00f00f00fULL;
    v = (v | v << 4) & 0x10c30c30c30c30c3ULL;
    v = (v | v << 2) & 0x1249249249249249ULL;
    return v;
}

inline uint64_t grid_coord(double x, double lo, double side) {
    double t = (x - lo) / side * (double)(1 << KEY_BITS);
    int64_t i = (int64_t)std::floor(t);
    if (i < 0) i = 0;
    if (i > (1 << KEY_BITS) - 1) i = (1 << KEY_BITS) - 1;
    return (uint64_t)i;
}

}  // namespace

extern "C" {

// posm: N x 4 float32 (x, y, z, m) in the caller's order; m is ignored here.
void* bh_build(int64_t n, const float* posm, int n_leaf, int n_grp) {
    if (n <= 0 || n > 0x7fffffff || n_leaf < 1 || n_grp < 1) return nullptr;
    Tree* t = new Tree;
    t->n = n; t->n_leaf = n_leaf; t->n_grp = n_grp;
    // O1 root cell
    double lo[3], hi[3];
    for (int a = 0; a < 3; ++a) { lo[a] = hi[a] = (double)posm[a]; }
    for (int64_t i = 1; i < n; ++i)
        for (int a = 0; a < 3; ++a) {
            double v = (double)posm[4 * i + a];
            if (v < lo[a]) lo[a] = v;
            if (v > hi[a]) hi[a] = v;
        }
    double ext = 0;
    for (int a = 0; a < 3; ++a) { t->root_c[a] = 0.5 * (lo[a] + hi[a]); ext = std::max(ext, hi[a] - lo[a]); }
    if (!(ext > 0)) ext = 1.0;
    t->root_side = ext * (1.0 + 1.0 / 1024.0);
    const double side = t->root_side;
    double rlo[3];
    for (int a = 0; a < 3; ++a) rlo[a] = t->root_c[a] - 0.5 * side;
    // O2 keys + stable sort
    std::vector<std::pair<uint64_t, int32_t>> kv((size_t)n);
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        uint64_t ix = grid_coord((double)posm[4 * i + 0], rlo[0], side);
        uint64_t iy = grid_coord((double)posm[4 * i + 1], rlo[1], side);
        uint64_t iz = grid_coord((double)posm[4 * i + 2], rlo[2], side);
        kv[(size_t)i] = {(spread3(ix) << 2) | (spread3(iy) << 1) | spread3(iz), (int32_t)i};
    }
#ifdef _OPENMP
    __gnu_parallel::sort(kv.begin(), kv.end());   // pairs: ties broken by original index => stable
#else
    std::sort(kv.begin(), kv.end());
#endif
    t->key.resize((size_t)n); t->perm.resize((size_t)n); t->pos.resize((size_t)n * 3);
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        t->key[(size_t)i] = kv[(size_t)i].first;
        int32_t o = kv[(size_t)i].second;
        t->perm[(size_t)i] = o;
        for (int a = 0; a < 3; ++a) t->pos[(size_t)i * 3 + a] = (double)posm[4 * (int64_t)o + a];
    }
    kv.clear(); kv.shrink_to_fit();
    // O2 cells, level by level from the top
    auto push_cell = [&](int32_t first, int32_t cnt, int lev, double cx, double cy, double cz, double s) {
        t->cell.push_back({first, cnt, 0, 0});
        t->geom.push_back(cx); t->geom.push_back(cy); t->geom.push_back(cz); t->geom.push_back(s);
        t->level.push_back(lev);
    };
    push_cell(0, (int32_t)n, 0, t->root_c[0], t->root_c[1], t->root_c[2], side);
    t->level_first.push_back(0);
    size_t lev_begin = 0;
    for (int lev = 0; lev <= KEY_BITS; ++lev) {
        size_t lev_end = t->cell.size();
        t->level_first.push_back((int32_t)lev_end);
        if (lev == KEY_BITS) break;
        const int shift = 3 * (KEY_BITS - 1 - lev);
        for (size_t c = lev_begin; c < lev_end; ++c) {
            Cell cc = t->cell[c];
            if (cc.n_ptcl <= n_leaf) continue;  // leaf
            const double cx = t->geom[4 * c], cy = t->geom[4 * c + 1], cz = t->geom[4 * c + 2], s = t->geom[4 * c + 3];
            const uint64_t* kb = t->key.data() + cc.first_ptcl;
            const uint64_t* ke = kb + cc.n_ptcl;
            int32_t first_child = (int32_t)t->cell.size();
            int n_child = 0;
            const uint64_t* p = kb;
            for (int oct = 0; oct < 8; ++oct) {
                // first key whose digit at this level exceeds oct
                const uint64_t* q = std::partition_point(p, ke, [&](uint64_t k) { return (int)((k >> shift) & 7) <= oct; });
                if (q > p) {
                    double hs = 0.5 * s, qs = 0.25 * s;
                    push_cell((int32_t)(cc.first_ptcl + (p - kb)), (int32_t)(q - p), lev + 1,
                              (oct & 4) ? cx + qs : cx - qs, (oct & 2) ? cy + qs : cy - qs, (oct & 1) ? cz + qs : cz - qs, hs);
                    ++n_child;
                }
                p = q;
            }
            t->cell[c].first_child = first_child;
            t->cell[c].n_child = n_child;
        }
        lev_begin = lev_end;
        if (t->cell.size() == lev_end) break;  // no deeper level
    }
    if (t->level_first.back() != (int32_t)t->cell.size()) t->level_first.push_back((int32_t)t->cell.size());
    // O3 groups: first cell on each root path with <= n_grp particles (or a leaf), Morton order
    std::vector<int32_t> stack;
    stack.push_back(0);
    while (!stack.empty()) {
        int32_t c = stack.back(); stack.pop_back();
        const Cell& cc = t->cell[(size_t)c];
        if (cc.n_ptcl <= n_grp || cc.n_child == 0) {
            t->grp_cell.push_back(c); t->grp_first.push_back(cc.first_ptcl); t->grp_n.push_back(cc.n_ptcl);
        } else {
            for (int k = cc.n_child - 1; k >= 0; --k) stack.push_back(cc.first_child + k);
        }
    }
    return t;
}

void bh_free(void* h) { delete (Tree*)h; }
int64_t bh_n_cell(void* h) { return (int64_t)((Tree*)h)->cell.size(); }
int64_t bh_n_group(void* h) { return (int64_t)((Tree*)h)->grp_first.size(); }
int32_t bh_n_level(void* h) { return (int32_t)((Tree*)h)->level_first.size() - 1; }

void bh_get_tree(void* h, int32_t* perm, int32_t* cells4, double* geom4, int32_t* level, int32_t* level_first, double* root4) {
    Tree* t = (Tree*)h;
    if (perm) std::memcpy(perm, t->perm.data(), t->perm.size() * sizeof(int32_t));
    if (cells4) std::memcpy(cells4, t->cell.data(), t->cell.size() * sizeof(Cell));
    if (geom4) std::memcpy(geom4, t->geom.data(), t->geom.size() * sizeof(double));
    if (level) std::memcpy(level, t->level.data(), t->level.size() * sizeof(int32_t));
    if (level_first) std::memcpy(level_first, t->level_first.data(), t->level_first.size() * sizeof(int32_t));
    if (root4) { root4[0] = t->root_c[0]; root4[1] = t->root_c[1]; root4[2] = t->root_c[2]; root4[3] = t->root_side; }
}

void bh_get_groups(void* h, int32_t* grp_cell, int32_t* grp_first, int32_t* grp_n) {
    Tree* t = (Tree*)h;
    size_t b = t->grp_first.size() * sizeof(int32_t);
    if (grp_cell) std::memcpy(grp_cell, t->grp_cell.data(), b);
    if (grp_first) std::memcpy(grp_first, t->grp_first.data(), b);
    if (grp_n) std::memcpy(grp_n, t->grp_n.data(), b);
}

// O4: one walk per group.  Returns totals through e_epj/e_spj; offsets are (n_group+1) int64.
int bh_build_lists(void* h, double theta, int64_t* epj_off, int64_t* spj_off, int64_t* e_epj, int64_t* e_spj) {
    Tree* t = (Tree*)h;
    if (!(theta >= 0)) return -1;
    const int64_t ng = (int64_t)t->grp_first.size();
    const int64_t BLK = 64;
    const int64_t nblk = (ng + BLK - 1) / BLK;
    t->blk_groups = BLK;
    t->blk_epj.assign((size_t)nblk, {});
    t->blk_spj.assign((size_t)nblk, {});
    t->epj_off.assign((size_t)ng + 1, 0);
    t->spj_off.assign((size_t)ng + 1, 0);
    const double th2 = theta * theta;
#pragma omp parallel
    {
        std::vector<int32_t> stack;
#pragma omp for schedule(dynamic, 1)
        for (int64_t b = 0; b < nblk; ++b) {
            std::vector<int32_t>& ve = t->blk_epj[(size_t)b];
            std::vector<int32_t>& vs = t->blk_spj[(size_t)b];
            for (int64_t g = b * BLK; g < std::min(ng, (b + 1) * BLK); ++g) {
                const int32_t f = t->grp_first[(size_t)g], cnt = t->grp_n[(size_t)g];
                double lo[3], hi[3];
                for (int a = 0; a < 3; ++a) lo[a] = hi[a] = t->pos[(size_t)f * 3 + a];
                for (int32_t i = f + 1; i < f + cnt; ++i)
                    for (int a = 0; a < 3; ++a) {
                        double v = t->pos[(size_t)i * 3 + a];
                        if (v < lo[a]) lo[a] = v;
                        if (v > hi[a]) hi[a] = v;
                    }
                const size_t e0 = ve.size(), s0 = vs.size();
                stack.clear();
                stack.push_back(0);
                while (!stack.empty()) {
                    const int32_t c = stack.back(); stack.pop_back();
                    const double* gm = &t->geom[(size_t)c * 4];
                    double d2 = 0;
                    for (int a = 0; a < 3; ++a) {
                        double s = gm[a], d = 0;
                        if (s < lo[a]) d = lo[a] - s;
                        else if (s > hi[a]) d = s - hi[a];
                        d2 += d * d;
                    }
                    const Cell& cc = t->cell[(size_t)c];
                    if (gm[3] * gm[3] > th2 * d2) {  // open iff l > theta * d
                        if (cc.n_child == 0) {
                            for (int32_t i = cc.first_ptcl; i < cc.first_ptcl + cc.n_ptcl; ++i) ve.push_back(i);
                        } else {
                            for (int k = cc.n_child - 1; k >= 0; --k) stack.push_back(cc.first_child + k);
                        }
                    } else {
                        vs.push_back(c);
                    }
                }
                t->epj_off[(size_t)g + 1] = (int64_t)(ve.size() - e0);
                t->spj_off[(size_t)g + 1] = (int64_t)(vs.size() - s0);
            }
        }
    }
    for (int64_t g = 0; g < ng; ++g) {
        t->epj_off[(size_t)g + 1] += t->epj_off[(size_t)g];
        t->spj_off[(size_t)g + 1] += t->spj_off[(size_t)g];
    }
    std::memcpy(epj_off, t->epj_off.data(), ((size_t)ng + 1) * sizeof(int64_t));
    std::memcpy(spj_off, t->spj_off.data(), ((size_t)ng + 1) * sizeof(int64_t));
    *e_epj = t->epj_off[(size_t)ng];
    *e_spj = t->spj_off[(size_t)ng];
    return 0;
}

// Short-range neighbour search ("we still use treewalk but with cell-opening criterion different from the
// standard opening angle", reading S24 of DESIGN.md).  hsml: smoothing length per
// particle in the CALLER's order (as posm was given to bh_build).  With R = 2 (1 + skin) x the largest h among a
// set of particles, cell c is opened for group g iff the gap between c's cube and g's particle box is <= max(R_g, R_c)
// (gather and scatter neighbours: a pair interacts when r < 2 max(h_i, h_k)); an opened leaf contributes its particles
// as EPJ, everything else is dropped -- there are no SPJ.  Purely geometric: no kernel arithmetic here.
int bh_build_neighbour_lists(void* h, const float* hsml, double skin, int64_t* epj_off, int64_t* spj_off, int64_t* e_epj) {
    Tree* t = (Tree*)h;
    if (!hsml || !(skin >= 0)) return -1;
    const int64_t ng = (int64_t)t->grp_first.size();
    const int64_t nc = (int64_t)t->cell.size();
    const double reach = 2.0 * (1.0 + skin);
    std::vector<double> hs((size_t)t->n), cell_h((size_t)nc, 0.0);
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < t->n; ++i) hs[(size_t)i] = (double)hsml[t->perm[(size_t)i]];
    for (int64_t c = nc - 1; c >= 0; --c) {  // children sit behind their parent: bottom-up in one reverse sweep
        const Cell& cc = t->cell[(size_t)c];
        double m = 0;
        if (cc.n_child == 0) {
            for (int32_t i = cc.first_ptcl; i < cc.first_ptcl + cc.n_ptcl; ++i) m = std::max(m, hs[(size_t)i]);
        } else {
            for (int k = 0; k < cc.n_child; ++k) m = std::max(m, cell_h[(size_t)(cc.first_child + k)]);
        }
        cell_h[(size_t)c] = m;
    }
    const int64_t BLK = 64;
    const int64_t nblk = (ng + BLK - 1) / BLK;
    t->blk_groups = BLK;
    t->blk_epj.assign((size_t)nblk, {});
    t->blk_spj.assign((size_t)nblk, {});
    t->epj_off.assign((size_t)ng + 1, 0);
    t->spj_off.assign((size_t)ng + 1, 0);
#pragma omp parallel
    {
        std::vector<int32_t> stack;
#pragma omp for schedule(dynamic, 1)
        for (int64_t b = 0; b < nblk; ++b) {
            std::vector<int32_t>& ve = t->blk_epj[(size_t)b];
            for (int64_t g = b * BLK; g < std::min(ng, (b + 1) * BLK); ++g) {
                const int32_t f = t->grp_first[(size_t)g], cnt = t->grp_n[(size_t)g];
                double lo[3], hi[3], hg = 0;
                for (int a = 0; a < 3; ++a) lo[a] = hi[a] = t->pos[(size_t)f * 3 + a];
                for (int32_t i = f; i < f + cnt; ++i) {
                    hg = std::max(hg, hs[(size_t)i]);
                    for (int a = 0; a < 3; ++a) {
                        double v = t->pos[(size_t)i * 3 + a];
                        if (v < lo[a]) lo[a] = v;
                        if (v > hi[a]) hi[a] = v;
                    }
                }
                const double rg = reach * hg;
                const size_t e0 = ve.size();
                stack.clear();
                stack.push_back(0);
                while (!stack.empty()) {
                    const int32_t c = stack.back(); stack.pop_back();
                    const double* gm = &t->geom[(size_t)c * 4];
                    const double half = 0.5 * gm[3];
                    double d2 = 0;
                    for (int a = 0; a < 3; ++a) {
                        double d = 0;
                        if (gm[a] + half < lo[a]) d = lo[a] - (gm[a] + half);
                        else if (gm[a] - half > hi[a]) d = (gm[a] - half) - hi[a];
                        d2 += d * d;
                    }
                    const double rc = reach * cell_h[(size_t)c];
                    const double r = rg > rc ? rg : rc;
                    if (!(d2 <= r * r)) continue;
                    const Cell& cc = t->cell[(size_t)c];
                    if (cc.n_child == 0) {
                        for (int32_t i = cc.first_ptcl; i < cc.first_ptcl + cc.n_ptcl; ++i) ve.push_back(i);
                    } else {
                        for (int k = cc.n_child - 1; k >= 0; --k) stack.push_back(cc.first_child + k);
                    }
                }
                t->epj_off[(size_t)g + 1] = (int64_t)(ve.size() - e0);
            }
        }
    }
    for (int64_t g = 0; g < ng; ++g) t->epj_off[(size_t)g + 1] += t->epj_off[(size_t)g];
    std::memcpy(epj_off, t->epj_off.data(), ((size_t)ng + 1) * sizeof(int64_t));
    std::memcpy(spj_off, t->spj_off.data(), ((size_t)ng + 1) * sizeof(int64_t));
    *e_epj = t->epj_off[(size_t)ng];
    return 0;
}

// Copies the lists built by bh_build_lists into caller arrays and releases the internal blocks.
void bh_get_lists(void* h, int32_t* epj_id, int32_t* spj_id) {
    Tree* t = (Tree*)h;
    const int64_t ng = (int64_t)t->grp_first.size();
    const int64_t BLK = t->blk_groups;
    const int64_t nblk = (int64_t)t->blk_epj.size();
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t b = 0; b < nblk; ++b) {
        const int64_t g0 = b * BLK;
        (void)ng;
        std::vector<int32_t>& ve = t->blk_epj[(size_t)b];
        std::vector<int32_t>& vs = t->blk_spj[(size_t)b];
        if (!ve.empty()) std::memcpy(epj_id + t->epj_off[(size_t)g0], ve.data(), ve.size() * sizeof(int32_t));
        if (!vs.empty()) std::memcpy(spj_id + t->spj_off[(size_t)g0], vs.data(), vs.size() * sizeof(int32_t));
        std::vector<int32_t>().swap(ve);
        std::vector<int32_t>().swap(vs);
    }
    t->blk_epj.clear(); t->blk_spj.clear();
}

// Method G1's host-side packing (Fig. 2 "DispatchKernelStream" copies EPJ and SPJ data per walk):
// for groups [g0, g1) write the records of their EPJ ids (from posm) and then of their SPJ ids (from spj, one
// float4 per cell) contiguously into out, and the run offsets (in records, relative to out) into joff[g1 - g0 + 1].
// A pure gather: no arithmetic.  OpenMP over groups.
void bh_pack_data_lists(int64_t g0, int64_t g1, const float* posm, const float* spj, const int64_t* epj_off, const int32_t* epj_id,
                        const int64_t* spj_off, const int32_t* spj_id, float* out, int64_t* joff) {
    joff[0] = 0;
    for (int64_t g = g0; g < g1; ++g) joff[g - g0 + 1] = joff[g - g0] + (epj_off[g + 1] - epj_off[g]) + (spj_off[g + 1] - spj_off[g]);
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t g = g0; g < g1; ++g) {
        float* o = out + 4 * joff[g - g0];
        for (int64_t k = epj_off[g]; k < epj_off[g + 1]; ++k, o += 4) std::memcpy(o, posm + 4 * (int64_t)epj_id[k], 16);
        for (int64_t k = spj_off[g]; k < spj_off[g + 1]; ++k, o += 4) std::memcpy(o, spj + 4 * (int64_t)spj_id[k], 16);
    }
}

}  // extern "C"
