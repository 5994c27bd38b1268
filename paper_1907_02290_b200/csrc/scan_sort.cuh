// Device-wide exclusive scan and stable LSD radix sort for the device-side construction step
// (paper: "radix sort of key-index pairs", 8-bit digits x 8 passes on
// 64-bit Morton keys).  Hand-written for sm_100a; no CUB / Thrust on this path.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace mwf {

// ---------------------------------------------------------------------------------------------------
// Exclusive scan, in place, of n elements (T = int32_t or int64_t).  Three-level recursion: every block
// scans SCAN_TILE elements and emits its total; the totals are scanned recursively; offsets are added back.
// `scratch` must hold scan_scratch_elems(n) elements of T.  Scanning n + 1 elements whose last input is
// zero leaves the grand total in data[n] (how every caller here obtains it).
constexpr int SCAN_THREADS = 512;
constexpr int SCAN_ITEMS = 8;
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_ITEMS;

inline int64_t scan_scratch_elems(int64_t n) {
    int64_t total = 0;
    while (n > 1) {
        n = (n + SCAN_TILE - 1) / SCAN_TILE;
        total += n + 1;
        if (n == 1) break;
    }
    return total + 2;
}

template <typename T>
__global__ void __launch_bounds__(SCAN_THREADS) k_scan_tiles(T* __restrict__ data, int64_t n, T* __restrict__ tile_sums) {
    __shared__ T s_warp[SCAN_THREADS / 32];
    const int64_t base = (int64_t)blockIdx.x * SCAN_TILE + (int64_t)threadIdx.x * SCAN_ITEMS;
    T v[SCAN_ITEMS];
    T sum = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        v[k] = (base + k < n) ? data[base + k] : T(0);
        sum += v[k];
    }
    // inclusive warp scan of the per-thread sums
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    T incl = sum;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const T up = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += up;
    }
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    if (warp == 0) {
        T w = (lane < SCAN_THREADS / 32) ? s_warp[lane] : T(0);
        T wi = w;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const T up = __shfl_up_sync(0xffffffffu, wi, d);
            if (lane >= d) wi += up;
        }
        if (lane < SCAN_THREADS / 32) s_warp[lane] = wi - w;  // exclusive prefix of the warps
        if (lane == SCAN_THREADS / 32 - 1 && tile_sums) tile_sums[blockIdx.x] = wi;
    }
    __syncthreads();
    T run = s_warp[warp] + incl - sum;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        if (base + k < n) data[base + k] = run;
        run += v[k];
    }
}

template <typename T>
__global__ void __launch_bounds__(SCAN_THREADS) k_scan_add(T* __restrict__ data, int64_t n, const T* __restrict__ tile_offsets) {
    const T off = tile_offsets[blockIdx.x];
    const int64_t base = (int64_t)blockIdx.x * SCAN_TILE + (int64_t)threadIdx.x * SCAN_ITEMS;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k)
        if (base + k < n) data[base + k] += off;
}

template <typename T>
cudaError_t scan_exclusive(T* data, int64_t n, T* scratch, cudaStream_t s) {
    if (n <= 0) return cudaSuccess;
    const int64_t nb = (n + SCAN_TILE - 1) / SCAN_TILE;
    if (nb == 1) {
        k_scan_tiles<T><<<1, SCAN_THREADS, 0, s>>>(data, n, nullptr);
        return cudaGetLastError();
    }
    k_scan_tiles<T><<<(unsigned)nb, SCAN_THREADS, 0, s>>>(data, n, scratch);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    e = scan_exclusive<T>(scratch, nb, scratch + nb + 1, s);
    if (e != cudaSuccess) return e;
    k_scan_add<T><<<(unsigned)nb, SCAN_THREADS, 0, s>>>(data, n, scratch);
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------------
// Stable LSD radix sort of (uint64 key, int32 value) pairs, 8-bit digits.  Per pass:
//   k_radix_hist     every block counts the digits of its tile of SORT_TILE consecutive pairs
//   scan_exclusive   over the digit-major table hist[digit * n_blocks + block]
//   k_radix_scatter  every block ranks its tile stably (warp match + per-warp counters), sorts it locally in
//                    shared memory so that equal digits leave as contiguous runs, and writes the runs out
constexpr int SORT_THREADS = 256;
constexpr int SORT_ITEMS = 8;
constexpr int SORT_TILE = SORT_THREADS * SORT_ITEMS;  // 2048 pairs = 24 KB of shared memory
constexpr int SORT_WARPS = SORT_THREADS / 32;

inline int64_t sort_blocks(int64_t n) { return (n + SORT_TILE - 1) / SORT_TILE; }

static __global__ void __launch_bounds__(SORT_THREADS) k_radix_hist(const uint64_t* __restrict__ keys, int64_t n, int shift, int32_t* __restrict__ hist,
                                                              int64_t n_blocks) {
    __shared__ int32_t s_hist[256];
    s_hist[threadIdx.x] = 0;
    __syncthreads();
    const int64_t base = (int64_t)blockIdx.x * SORT_TILE;
#pragma unroll
    for (int k = 0; k < SORT_ITEMS; ++k) {
        const int64_t i = base + k * SORT_THREADS + threadIdx.x;
        if (i < n) atomicAdd(&s_hist[(int)((keys[i] >> shift) & 255)], 1);
    }
    __syncthreads();
    hist[(int64_t)threadIdx.x * n_blocks + blockIdx.x] = s_hist[threadIdx.x];
}

static __global__ void __launch_bounds__(SORT_THREADS) k_radix_scatter(const uint64_t* __restrict__ keys_in, const int32_t* __restrict__ vals_in,
                                                                 uint64_t* __restrict__ keys_out, int32_t* __restrict__ vals_out, int64_t n, int shift,
                                                                 const int32_t* __restrict__ hist_scanned, int64_t n_blocks) {
    __shared__ int32_t s_cnt[SORT_WARPS][256];   // per-warp digit counters, then running local offsets
    __shared__ int32_t s_local[256];             // first local slot of each digit in the sorted tile
    __shared__ int32_t s_global[256];            // first global slot of each digit for this block
    __shared__ uint64_t s_keys[SORT_TILE];
    __shared__ int32_t s_vals[SORT_TILE];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t base = (int64_t)blockIdx.x * SORT_TILE;
    const int tile_n = (int)((n - base) < SORT_TILE ? (n - base) : SORT_TILE);
    for (int k = threadIdx.x; k < SORT_WARPS * 256; k += SORT_THREADS) (&s_cnt[0][0])[k] = 0;
    __syncthreads();
    // warp w owns the consecutive pairs [w * 256, (w + 1) * 256) of the tile, in chunks of 32
    uint64_t key[SORT_ITEMS];
    int32_t val[SORT_ITEMS];
    int dig[SORT_ITEMS];
#pragma unroll
    for (int k = 0; k < SORT_ITEMS; ++k) {
        const int t = warp * (32 * SORT_ITEMS) + k * 32 + lane;
        const bool in = t < tile_n;
        key[k] = in ? keys_in[base + t] : ~0ULL;
        val[k] = in ? vals_in[base + t] : 0;
        dig[k] = in ? (int)((key[k] >> shift) & 255) : 256;  // 256: padding, never counted
        const unsigned peers = __match_any_sync(0xffffffffu, dig[k]);
        if (in && lane == __ffs(peers) - 1) s_cnt[warp][dig[k]] += __popc(peers);
        __syncwarp();
    }
    __syncthreads();
    // exclusive prefix over (digit, warp): local slot where each warp's run of each digit starts
    {
        const int d = threadIdx.x;
        int32_t tot = 0;
#pragma unroll
        for (int w = 0; w < SORT_WARPS; ++w) {
            const int32_t c = s_cnt[w][d];
            s_cnt[w][d] = tot;
            tot += c;
        }
        // block-wide exclusive scan of the digit totals
        int32_t incl = tot;
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            const int32_t up = __shfl_up_sync(0xffffffffu, incl, off);
            if (lane >= off) incl += up;
        }
        __shared__ int32_t s_wsum[SORT_WARPS];
        if (lane == 31) s_wsum[warp] = incl;
        __syncthreads();
        int32_t wbase = 0;
#pragma unroll
        for (int w = 0; w < SORT_WARPS; ++w)
            if (w < warp) wbase += s_wsum[w];
        s_local[d] = wbase + incl - tot;
        s_global[d] = hist_scanned[(int64_t)d * n_blocks + blockIdx.x];
    }
    __syncthreads();
    // stable local rank -> sorted tile in shared memory
#pragma unroll
    for (int k = 0; k < SORT_ITEMS; ++k) {
        const bool in = dig[k] < 256;
        const unsigned peers = __match_any_sync(0xffffffffu, dig[k]);
        int slot = 0;
        if (in) slot = s_local[dig[k]] + s_cnt[warp][dig[k]] + __popc(peers & ((1u << lane) - 1u));
        __syncwarp();
        if (in && lane == __ffs(peers) - 1) s_cnt[warp][dig[k]] += __popc(peers);
        __syncwarp();
        if (in) {
            s_keys[slot] = key[k];
            s_vals[slot] = val[k];
        }
    }
    __syncthreads();
    // write out: consecutive threads hold consecutive slots, equal digits go to consecutive global slots
    for (int t = threadIdx.x; t < tile_n; t += SORT_THREADS) {
        const uint64_t kk = s_keys[t];
        const int d = (int)((kk >> shift) & 255);
        const int64_t dst = (int64_t)s_global[d] + (t - s_local[d]);
        keys_out[dst] = kk;
        vals_out[dst] = s_vals[t];
    }
}

// Sorts n pairs; result ends in (keys_a, vals_a) (8 passes: an even number of ping-pongs).  hist must hold
// 256 * sort_blocks(n) + 1 int32, scratch scan_scratch_elems(256 * sort_blocks(n) + 1) int32.
inline cudaError_t radix_sort_pairs(uint64_t* keys_a, int32_t* vals_a, uint64_t* keys_b, int32_t* vals_b, int64_t n, int key_bits,
                                    int32_t* hist, int32_t* scratch, cudaStream_t s) {
    if (n <= 0) return cudaSuccess;
    const int64_t nb = sort_blocks(n);
    int passes = (key_bits + 7) / 8;
    if (passes & 1) ++passes;  // even, so that the result lands in the `a` buffers
    for (int p = 0; p < passes; ++p) {
        const int shift = 8 * p;
        uint64_t* ki = (p & 1) ? keys_b : keys_a;
        uint64_t* ko = (p & 1) ? keys_a : keys_b;
        int32_t* vi = (p & 1) ? vals_b : vals_a;
        int32_t* vo = (p & 1) ? vals_a : vals_b;
        k_radix_hist<<<(unsigned)nb, SORT_THREADS, 0, s>>>(ki, n, shift, hist, nb);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
        e = scan_exclusive<int32_t>(hist, 256 * nb, scratch, s);
        if (e != cudaSuccess) return e;
        k_radix_scatter<<<(unsigned)nb, SORT_THREADS, 0, s>>>(ki, vi, ko, vo, n, shift, hist, nb);
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

}  // namespace mwf
