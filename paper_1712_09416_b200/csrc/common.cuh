// common.cuh -- device-side views, constants and small helpers of the sm_100a tracker.
// Layouts are described in DESIGN.md "Data layout in HBM".
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "tpctrack.h"

namespace tpc {

constexpr int kCellPad = 32;          // cell table of a bin holds up to n_hits + kCellPad entries
constexpr float kGridPad = 1.0e-3f;   // cm added to every grid query so that rounding never hides a candidate
constexpr int kChunk = 32;            // tracklets per table chunk: table[chunk][row][lane]

// error bits raised by kernels
constexpr unsigned kErrBadRow = 1u, kErrRowCapacity = 2u, kErrSeedCapacity = 4u;

// device counters (unsigned long long each)
enum { CNT_ERR = 0, CNT_LINKS, CNT_ROW_VISITS, CNT_TL_HITS, CNT_TRACKS, CNT_TRACK_HITS, CNT_N };

// One event's input arrays (device pointers) and its place in the batch-global cluster numbering.
struct EventSrc {
    const float* y;
    const float* z;
    const int32_t* row;
    int32_t n;
    int32_t off;
};

// Constants of a tracker, passed by value to the kernels (lands in the constant bank).
struct Const {
    float row_x[TPC_MAX_ROWS + 1];
    int32_t n_sectors, n_rows;
    float tan_half_angle, sigma_y2, sigma_z2, kB;
    tpc_params p;
};

// Everything a kernel may touch, for one batch.
struct View {
    int32_t n_events, n_tasks, n_bins, N;
    const EventSrc* ev;      // [n_events]
    const int32_t* sec_off;  // [n_events][n_sectors+1] event-local
    // K1: bucket by (task,row), sort by grid cell
    int32_t* bin_count;      // [n_bins+1]
    int32_t* bin_start;      // [n_bins+1] exclusive scan of bin_count
    uint16_t* slot;          // [N] position of a cluster inside its bin, arrival order (batch-global cluster order)
    float* ty; float* tz; int32_t* tidx; // [N] bucketed, unsorted
    float* sy; float* sz; int32_t* sorig; // [N] sorted by (task,row,cell,index); sorig = caller's index in its event
    float4* grid_f;          // [n_bins] y0, z0, 1/dy, 1/dz
    int2* grid_n;            // [n_bins] ny, nz
    uint16_t* cells;         // [N + n_bins*kCellPad] first hit of each cell, relative to bin_start
    // K2-K4
    int32_t *link_up, *link_dn, *clink_up, *clink_dn; // [N] batch-global sorted index or -1
    int32_t* seed_count;     // [n_bins+1]
    int32_t* seed_start;     // [n_bins+1]
    int32_t* seeds;          // [S_cap] sorted index of the start hit, canonical order
    int32_t* seed_bin;       // [S_cap]
    int32_t S_cap;
    // K5
    int32_t* tl_table;       // [S_cap/32][n_rows][32] sorted index or -1
    int32_t* tl_rows;        // [S_cap] first_row | last_row << 8 | n_hits << 16
    float* tl_par;           // [6][S_cap] y z s t q chi2
    // K6
    uint32_t* owner;         // [N] best key among tracklets holding the hit
    int32_t* tl_nown;        // [S_cap+1] hits owned (0 when the track is dropped)
    int32_t* tl_keep;        // [S_cap+1] 1 when the track is kept
    int32_t* trk_scan;       // [S_cap+1]
    int32_t* hit_scan;       // [S_cap+1]
    int32_t* ev_off;         // [2][n_events+1] track / hit offsets of each event
    // outputs
    int32_t *o_sector, *o_first_hit, *o_n_hits, *o_ndf, *o_hit_idx;
    float *o_x, *o_y, *o_z, *o_sinphi, *o_tgl, *o_qpt, *o_chi2;
    unsigned long long* cnt; // [CNT_N]
};

__device__ __forceinline__ int lane_id() { return threadIdx.x & 31; }

// Row grid of one bin.
struct RowGrid {
    float y0, z0, idy, idz;
    int ny, nz;
    int base;              // bin_start
    const uint16_t* cs;    // cell table of this bin
    __device__ __forceinline__ int cy(float y) const {
        int i = (int)((y - y0) * idy);
        return max(0, min(i, ny - 1));
    }
    __device__ __forceinline__ int cz(float z) const {
        int i = (int)((z - z0) * idz);
        return max(0, min(i, nz - 1));
    }
};

__device__ __forceinline__ RowGrid load_grid(const View& v, int bin) {
    RowGrid g;
    const float4 f = __ldg(&v.grid_f[bin]);
    const int2 n = __ldg(&v.grid_n[bin]);
    g.y0 = f.x; g.z0 = f.y; g.idy = f.z; g.idz = f.w; g.ny = n.x; g.nz = n.y;
    g.base = __ldg(&v.bin_start[bin]);
    g.cs = v.cells + (size_t)g.base + (size_t)bin * kCellPad;
    return g;
}

// Walks the hits of all cells overlapping [y-wy, y+wy] x [z-wz, z+wz] (padded); exact tests are the caller's.
struct GridIter {
    const uint16_t* cs;
    int base, ny, iy0, iy1, iz, iz1, p, pend;
    __device__ __forceinline__ void start(const RowGrid& g, float y, float z, float wy, float wz) {
        cs = g.cs; base = g.base; ny = g.ny;
        iy0 = g.cy(y - wy - kGridPad); iy1 = g.cy(y + wy + kGridPad);
        iz = g.cz(z - wz - kGridPad) - 1; iz1 = g.cz(z + wz + kGridPad);
        p = 0; pend = 0;
    }
    __device__ __forceinline__ bool next(int& h) {
        while (p >= pend) {
            if (++iz > iz1) return false;
            p = base + cs[iz * ny + iy0];
            pend = base + cs[iz * ny + iy1 + 1];
        }
        h = p++;
        return true;
    }
};

}  // namespace tpc
