// mwf_monopoles_static(): the bottom-up monopole pass (paper P:160, "multipole moments of all local tree cells are
// calculated, from the bottom to the top of the tree") for callers that are not allowed to allocate device memory.
//
// Who that is.  Every other entry point of libmwf.so lives behind an mwf_ctx, and a ctx needs an arena: either the
// library cudaMalloc's it, or the caller does (a torch tensor, say) and hands it over.  Some callers can do neither:
//   - a plugin inside a host application whose own pool already owns the device memory, so that a cudaMalloc from a
//     guest library may fail or is simply forbidden by the application's rules;
//   - a step function that runs inside somebody else's timed or latency-bound loop, where cudaMalloc / cudaFree stall
//     the whole device (both synchronise it) and a stall is worse than a size limit;
//   - code that runs late in a job on a nearly full GPU, when an allocation that worked in testing is the one call that
//     can fail.
// For them this file keeps the pass's working memory -- fp64 moments, parent links and arrival counters, 40 bytes per
// cell -- in ONE file-scope __device__ array of fixed size, MWF_STATIC_MAX_CELL cells (5 MiB).  It is part of the
// library image: every GPU on which the library's code is loaded carries it until the process exits, used or not, which is
// why the maximum is modest.  The entry point calls no cudaMalloc, no cudaFree and no library routine that allocates; the
// caller passes the inputs and the output, all already on the device.
//
// Host code cannot use the array's name as a pointer (on the host the name is only a handle for the runtime; a kernel
// given that value would fault or touch unrelated memory), so the first call on each device asks the runtime for the
// array's device address (cudaGetSymbolAddress, with that device current) and keeps it; kernels get that address as an
// argument.  That first call is therefore a set-up call: make it before any stream capture is begun.
//
// All calls on one GPU share the array and it keeps whatever the last call left.  What has to start from a known state
// (parent links, arrival counters) is reset on the caller's stream at the start of every call; the moments are always
// written before they are read.  Two calls that overlap on the same GPU (different streams, or two host threads) race on
// it: serialise them.
//
// The arithmetic is that of the climb variant in monopole_kernel.cu (leaf sums in fp64, the last child to arrive combines
// its siblings in child order, one rounding to float at the end), restated here so that no existing kernel or launch
// path changes.
#include <cuda_runtime.h>
#include <stdint.h>

#include <mutex>
#include <string>

#include "mwf.h"

namespace {

constexpr int64_t MAX_CELL = MWF_STATIC_MAX_CELL;
constexpr int MAX_DEVICE = 64;

// layout of the scratch array: [moments: double4 per cell][parent: int32 per cell][arrivals: int32 per cell]
constexpr size_t OFF_MOM = 0;
constexpr size_t OFF_PARENT = OFF_MOM + sizeof(double4) * MAX_CELL;
constexpr size_t OFF_ARRIVED = OFF_PARENT + sizeof(int32_t) * MAX_CELL;
constexpr size_t SCRATCH_BYTES = OFF_ARRIVED + sizeof(int32_t) * MAX_CELL;
static_assert(OFF_PARENT % 256 == 0 && OFF_ARRIVED % 256 == 0, "sub-arrays keep the 256-byte alignment");

static __device__ __align__(256) unsigned char g_static_scratch[SCRATCH_BYTES];

std::mutex g_mu;
void* g_scratch_addr[MAX_DEVICE];       // device address of g_static_scratch per device ordinal, 0 = not asked yet
thread_local std::string t_err;

// A cell's child range is followed only when it lies behind the cell and inside the array, its particle range only
// inside [0, n_ptcl): a malformed tree gives wrong numbers for the cells it touches, never an access outside the buffers.
__device__ __forceinline__ bool children_ok(const mwf_cell c, int64_t self, int64_t n_cell) {
    return c.n_child > 0 && c.n_child <= 8 && (int64_t)c.first_child > self && (int64_t)c.first_child + c.n_child <= n_cell;
}

__global__ void __launch_bounds__(256) k_static_parents(const mwf_cell* __restrict__ cells, int64_t n_cell, int32_t* __restrict__ parent) {
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= n_cell) return;
    const mwf_cell cc = cells[c];
    if (!children_ok(cc, c, n_cell)) return;
    for (int k = 0; k < cc.n_child; ++k) parent[cc.first_child + k] = (int32_t)c;
}

__device__ __forceinline__ void write_record(float4* __restrict__ spj, int64_t c, double sx, double sy, double sz, double m, float4 fallback) {
    float4 r;
    if (m > 0.0) {
        const double inv = 1.0 / m;
        r = make_float4((float)(sx * inv), (float)(sy * inv), (float)(sz * inv), (float)m);
    } else {  // massless cell: exerts nothing; keep a finite position
        r = make_float4(fallback.x, fallback.y, fallback.z, 0.f);
    }
    spj[c] = r;
}

__global__ void __launch_bounds__(128) k_static_monopoles(const mwf_cell* __restrict__ cells, int64_t n_cell, const float4* __restrict__ ptcl,
                                                          int64_t n_ptcl, float4* __restrict__ spj, double4* __restrict__ mom,
                                                          const int32_t* __restrict__ parent, int32_t* __restrict__ arrived) {
    const int64_t c0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c0 >= n_cell) return;
    const mwf_cell leaf = cells[c0];
    if (children_ok(leaf, c0, n_cell)) return;  // an internal cell is done by the last of its children to arrive
    int64_t lo = leaf.first_ptcl, hi = (int64_t)leaf.first_ptcl + leaf.n_ptcl;
    lo = lo < 0 ? 0 : lo;
    hi = hi > n_ptcl ? n_ptcl : hi;
    double sx = 0.0, sy = 0.0, sz = 0.0, m = 0.0;
    for (int64_t k = lo; k < hi; ++k) {
        const float4 q = ptcl[k];
        const double mq = (double)q.w;
        m += mq;
        sx += mq * (double)q.x;
        sy += mq * (double)q.y;
        sz += mq * (double)q.z;
    }
    mom[c0] = make_double4(sx, sy, sz, m);
    write_record(spj, c0, sx, sy, sz, m, lo < hi ? ptcl[lo] : make_float4(0.f, 0.f, 0.f, 0.f));
    int64_t c = c0;
    for (;;) {
        const int32_t par = parent[c];
        if (par < 0) break;  // the root, or a cell nobody claimed
        const mwf_cell pc = cells[par];
        __threadfence();  // this cell's moments are visible before its arrival is
        if (atomicAdd(&arrived[par], 1) != pc.n_child - 1) break;  // a later sibling carries on
        __threadfence();
        sx = sy = sz = m = 0.0;
        for (int k = 0; k < pc.n_child; ++k) {
            const double2* q = reinterpret_cast<const double2*>(&mom[pc.first_child + k]);
            const double2 a = __ldcg(q), b = __ldcg(q + 1);  // from L2: other SMs wrote them
            sx += a.x; sy += a.y; sz += b.x; m += b.y;
        }
        mom[par] = make_double4(sx, sy, sz, m);
        const bool in = pc.first_ptcl >= 0 && (int64_t)pc.first_ptcl < n_ptcl;
        write_record(spj, par, sx, sy, sz, m, in ? ptcl[pc.first_ptcl] : make_float4(0.f, 0.f, 0.f, 0.f));
        c = par;
    }
}

int fail_cuda(const char* what, cudaError_t e) {
    t_err = std::string(what) + ": " + cudaGetErrorString(e);
    return MWF_ECUDA;
}

}  // namespace

extern "C" int mwf_monopoles_static(const mwf_cell* cells, int64_t n_cell, const mwf_posm* ptcl, int64_t n_ptcl, mwf_posm* spj, void* stream) {
    t_err.clear();
    if (!cells || !ptcl || !spj || n_cell <= 0 || n_ptcl <= 0) {
        t_err = "mwf_monopoles_static: null pointer or non-positive size";
        return MWF_EINVAL;
    }
    if (n_cell > MAX_CELL) {
        t_err = "mwf_monopoles_static: n_cell = " + std::to_string(n_cell) + " exceeds MWF_STATIC_MAX_CELL = " + std::to_string(MAX_CELL) +
                " (the scratch is a fixed array in the library image; use an mwf_ctx for larger trees)";
        return MWF_ENOMEM;
    }
    if ((reinterpret_cast<uintptr_t>(cells) | reinterpret_cast<uintptr_t>(ptcl) | reinterpret_cast<uintptr_t>(spj)) & 15) {
        t_err = "mwf_monopoles_static: cells, ptcl and spj must be 16-byte aligned (they are read and written as 16-byte records)";
        return MWF_EINVAL;
    }
    if (n_ptcl > INT32_MAX) {
        t_err = "mwf_monopoles_static: n_ptcl exceeds the 32-bit particle indices of mwf_cell";
        return MWF_EINVAL;
    }
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail_cuda("cudaGetDevice", e);
    if (dev < 0 || dev >= MAX_DEVICE) {
        t_err = "mwf_monopoles_static: device ordinal beyond the table of " + std::to_string(MAX_DEVICE);
        return MWF_EINVAL;
    }
    unsigned char* base;
    {   // set-up, once per device, with that device current: the device address behind the host-side symbol
        std::lock_guard<std::mutex> lock(g_mu);
        if (!g_scratch_addr[dev]) {
            void* p = nullptr;
            if ((e = cudaGetSymbolAddress(&p, g_static_scratch)) != cudaSuccess) return fail_cuda("cudaGetSymbolAddress", e);
            g_scratch_addr[dev] = p;
        }
        base = static_cast<unsigned char*>(g_scratch_addr[dev]);
    }
    double4* mom = reinterpret_cast<double4*>(base + OFF_MOM);
    int32_t* parent = reinterpret_cast<int32_t*>(base + OFF_PARENT);
    int32_t* arrived = reinterpret_cast<int32_t*>(base + OFF_ARRIVED);
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    // the array still holds the last call's links and counts
    if ((e = cudaMemsetAsync(parent, 0xFF, (size_t)n_cell * sizeof(int32_t), s)) != cudaSuccess) return fail_cuda("cudaMemsetAsync", e);
    if ((e = cudaMemsetAsync(arrived, 0, (size_t)n_cell * sizeof(int32_t), s)) != cudaSuccess) return fail_cuda("cudaMemsetAsync", e);
    k_static_parents<<<(unsigned)((n_cell + 255) / 256), 256, 0, s>>>(cells, n_cell, parent);
    if ((e = cudaGetLastError()) != cudaSuccess) return fail_cuda("k_static_parents", e);
    k_static_monopoles<<<(unsigned)((n_cell + 127) / 128), 128, 0, s>>>(cells, n_cell, reinterpret_cast<const float4*>(ptcl), n_ptcl, reinterpret_cast<float4*>(spj), mom,
                                                                         parent, arrived);
    if ((e = cudaGetLastError()) != cudaSuccess) return fail_cuda("k_static_monopoles", e);
    return MWF_OK;
}

extern "C" const char* mwf_static_last_error(void) { return t_err.c_str(); }
