// scan.cuh -- exclusive prefix sum of int32 (out[0..n], out[n] = total) in three launches:
// per-tile totals, one-block scan of the totals, per-tile scan with the tile offset.
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

__global__ void __launch_bounds__(kScanThreads) k_scan_tile_totals(const int32_t* __restrict__ in, int n,
                                                                  int32_t* __restrict__ totals) {
    __shared__ int tot;
    const int base = blockIdx.x * kScanTile;
    int s = 0;
#pragma unroll
    for (int k = 0; k < kScanItems; k++) {
        int i = base + k * kScanThreads + threadIdx.x;
        if (i < n) s += in[i];
    }
    block_excl_scan<kScanThreads>(s, &tot);
    if (threadIdx.x == 0) totals[blockIdx.x] = tot;
}

// one block: exclusive scan of up to 1024*items totals in place
__global__ void __launch_bounds__(1024) k_scan_totals(int32_t* __restrict__ totals, int m) {
    __shared__ int tot;
    const int per = (m + 1023) / 1024;
    const int b = threadIdx.x * per;
    int s = 0;
    for (int k = 0; k < per; k++) if (b + k < m) s += totals[b + k];
    int ex = block_excl_scan<1024>(s, &tot);
    for (int k = 0; k < per; k++)
        if (b + k < m) { int v = totals[b + k]; totals[b + k] = ex; ex += v; }
    if (threadIdx.x == 0) totals[m] = tot;
}

__global__ void __launch_bounds__(kScanThreads) k_scan_apply(const int32_t* __restrict__ in, int n,
                                                            const int32_t* __restrict__ totals,
                                                            int32_t* __restrict__ out) {
    __shared__ int tot;
    __shared__ int tile[kScanTile];
    const int base = blockIdx.x * kScanTile;
    // blocked arrangement through shared memory so that global accesses stay coalesced
    for (int k = 0; k < kScanItems; k++) {
        int j = k * kScanThreads + threadIdx.x;
        tile[j] = (base + j < n) ? in[base + j] : 0;
    }
    __syncthreads();
    int v[kScanItems], s = 0;
#pragma unroll
    for (int k = 0; k < kScanItems; k++) { v[k] = tile[threadIdx.x * kScanItems + k]; s += v[k]; }
    int ex = block_excl_scan<kScanThreads>(s, &tot) + totals[blockIdx.x];
#pragma unroll
    for (int k = 0; k < kScanItems; k++) { tile[threadIdx.x * kScanItems + k] = ex; ex += v[k]; }
    __syncthreads();
    for (int k = 0; k < kScanItems; k++) {
        int j = k * kScanThreads + threadIdx.x;
        if (base + j < n) out[base + j] = tile[j];
    }
    if (blockIdx.x == gridDim.x - 1 && threadIdx.x == 0) out[n] = totals[gridDim.x];
}

// host: out[0..n] <- exclusive scan of in[0..n).  scratch needs n/kScanTile + 2 ints.  3 launches.
inline int scan_exclusive(const int32_t* in, int32_t* out, int n, int32_t* scratch, cudaStream_t st) {
    const int tiles = n > 0 ? (n + kScanTile - 1) / kScanTile : 1;
    k_scan_tile_totals<<<tiles, kScanThreads, 0, st>>>(in, n, scratch);
    k_scan_totals<<<1, 1024, 0, st>>>(scratch, tiles);
    k_scan_apply<<<tiles, kScanThreads, 0, st>>>(in, n, scratch, out);
    return 3;
}

}  // namespace tpc
