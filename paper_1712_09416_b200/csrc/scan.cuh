// scan.cuh -- exclusive prefix sum of int32 (out[0..n], out[n] = total) in ONE launch: tiles of 2048 elements,
// each tile publishes its sum at once and then looks back over the tiles before it until it meets one whose
// inclusive prefix is already known ("decoupled look-back").  Tiles take their number from a device counter, so
// a tile never waits for one that has not started.  The counter and the tiles' status words are cleared by one
// memset in front of the launch (no host-side state: the launch sequence can be captured in a CUDA graph).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace tpc {

constexpr int kScanThreads = 256;
constexpr int kScanItems = 8;
constexpr int kScanTile = kScanThreads * kScanItems;

__device__ __forceinline__ int warp_incl_scan(int v) {
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int t = __shfl_up_sync(0xffffffffu, v, o);
        if ((threadIdx.x & 31) >= o) v += t;
    }
    return v;
}

// exclusive scan of one value per thread across the block; returns the exclusive prefix, total in *total
template <int THREADS>
__device__ __forceinline__ int block_excl_scan(int v, int* total) {
    __shared__ int wsum[THREADS / 32];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    int inc = warp_incl_scan(v);
    if (lane == 31) wsum[w] = inc;
    __syncthreads();
    if (w == 0) {
        int s = lane < THREADS / 32 ? wsum[lane] : 0;
        int si = warp_incl_scan(s);
        if (lane < THREADS / 32) wsum[lane] = si - s;
        if (lane == THREADS / 32 - 1) *total = si;
    }
    __syncthreads();
    int r = inc - v + wsum[w];
    __syncthreads();
    return r;
}

// scratch[0] = tile counter, scratch[1 + t] = status of tile t: flag << 32 | value; flag 1 = tile sum, 2 = inclusive prefix
__global__ void __launch_bounds__(kScanThreads) k_scan(const int32_t* __restrict__ in, int n, int32_t* __restrict__ out,
                                                      unsigned long long* scratch) {
    __shared__ int tot, s_tile, s_prefix;
    __shared__ int tile[kScanTile];
    unsigned long long* const status = scratch + 1;
    if (threadIdx.x == 0) s_tile = (int)atomicAdd(scratch, 1ull);
    __syncthreads();
    const int t = s_tile, base = t * kScanTile;
    // blocked arrangement through shared memory so that global accesses stay coalesced
    for (int k = 0; k < kScanItems; k++) {
        const int j = k * kScanThreads + threadIdx.x;
        tile[j] = (base + j < n) ? in[base + j] : 0;
    }
    __syncthreads();
    int v[kScanItems], s = 0;
#pragma unroll
    for (int k = 0; k < kScanItems; k++) { v[k] = tile[threadIdx.x * kScanItems + k]; s += v[k]; }
    int ex = block_excl_scan<kScanThreads>(s, &tot);
    if (threadIdx.x < 32) {   // warp 0 publishes the tile's sum and looks back
        const int lane = threadIdx.x;
        volatile unsigned long long* st = status;
        int prefix = 0;
        if (t == 0) {
            if (lane == 0) { __threadfence(); st[0] = (2ull << 32) | (unsigned int)tot; }
        } else {
            if (lane == 0) { __threadfence(); st[t] = (1ull << 32) | (unsigned int)tot; }
            for (int j0 = t - 1; j0 >= 0; j0 -= 32) {   // 32 predecessors at a time, nearest first
                const int j = j0 - lane;
                unsigned long long w = 0;
                bool ready = j < 0;
                while (!__all_sync(0xffffffffu, ready)) {
                    if (!ready) { w = st[j]; ready = (w >> 32) != 0; }
                }
                const bool full = j >= 0 && (w >> 32) == 2;
                const unsigned fm = __ballot_sync(0xffffffffu, full);
                const int stop = fm ? __ffs(fm) - 1 : 31;         // the nearest tile that knows its inclusive prefix
                int part = (j >= 0 && lane <= stop) ? (int)(unsigned int)w : 0;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
                prefix += part;
                if (fm) break;
            }
            if (lane == 0) { __threadfence(); st[t] = (2ull << 32) | (unsigned int)(prefix + tot); }
        }
        if (lane == 0) s_prefix = prefix;
    }
    __syncthreads();
    ex += s_prefix;
#pragma unroll
    for (int k = 0; k < kScanItems; k++) { tile[threadIdx.x * kScanItems + k] = ex; ex += v[k]; }
    __syncthreads();
    for (int k = 0; k < kScanItems; k++) {
        const int j = k * kScanThreads + threadIdx.x;
        if (base + j < n) out[base + j] = tile[j];
    }
    if (t == (int)gridDim.x - 1 && threadIdx.x == 0) out[n] = s_prefix + tot;
}

// host: out[0..n] <- exclusive scan of in[0..n).  1 launch (+ 1 memset).  scratch: n / kScanTile + 2 words of 8 bytes.
inline int scan_exclusive(const int32_t* in, int32_t* out, int n, unsigned long long* scratch, cudaStream_t st) {
    const int tiles = n > 0 ? (n + kScanTile - 1) / kScanTile : 1;
    cudaMemsetAsync(scratch, 0, sizeof(unsigned long long) * (size_t)(tiles + 1), st);
    k_scan<<<tiles, kScanThreads, 0, st>>>(in, n, out, scratch);
    return 1;
}

}  // namespace tpc
