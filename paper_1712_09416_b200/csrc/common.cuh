// common.cuh -- device-side views, constants and small helpers of the sm_100a tracker.
// Layouts are described in DESIGN.md "Data layout in HBM".
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "tpctrack.h"

namespace tpc {

#ifndef TPC_CELLS_PER_HIT
#define TPC_CELLS_PER_HIT 3
#endif
constexpr int kCellsPerHit = TPC_CELLS_PER_HIT;       // grid cells per hit of a bin (the cells are this much finer in y than in z)
constexpr int kCellPad = 32;          // cell table of a bin holds up to kCellsPerHit * n_hits + kCellPad entries
constexpr int kMaxCells = kCellsPerHit == 1 ? TPC_MAX_ROW_HITS + kCellPad - 1 : 4096;  // and never more than kMaxCells + 1
constexpr float kGridPad = 1.0e-3f;   // cm added to every grid query so that rounding never hides a candidate
constexpr uint16_t kNoHit = 0xffffu;  // empty entry of a tracklet's row -> hit table (hits are row-local, < 2048)
constexpr unsigned kFull = 0xffffffffu;

// error bits raised by kernels
constexpr unsigned kErrBadRow = 1u, kErrRowCapacity = 2u, kErrSeedCapacity = 4u, kErrHang = 8u, kErrSelCapacity = 16u,
                   kErrSlotCapacity = 32u,   // K5: more tracklets under way in a sector task than state slots
                   kErrBadInput = 64u;       // checked mode: non-finite y / z, or x off its pad row
constexpr unsigned kErrFatal = kErrBadRow | kErrRowCapacity | kErrBadInput;   // the later kernels do nothing after these

// the stages after K1 start with this: a batch that K1 has rejected is not worked on (its arrays may be incomplete)
// (a cached read: K1's bits were set by earlier kernels; a volatile one makes every warp of the grid queue at one L2 line)
#define TPC_RETURN_IF_REJECTED(v) do { if (__ldg(&(v).cnt[CNT_ERR]) & kErrFatal) return; } while (0)

// device counters (unsigned long long each)
constexpr int kNCursors = 4;           // work cursors: [0] K5 sector tasks, [2] refit
enum { CNT_ERR = 0, CNT_LINKS, CNT_ROW_VISITS, CNT_TL_HITS, CNT_TRACKS, CNT_TRACK_HITS, CNT_UPDATES, CNT_REFIT_VISITS, CNT_TRACKLETS, CNT_LARGE_BINS, CNT_PROF, CNT_N = CNT_PROF + 16 };

// One event's input arrays (device pointers) and its place in the batch-global cluster numbering.
struct EventSrc {
    const float* x;          // may be NULL; read in checked mode only
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
    float merge_cd, merge_sd;   // cos, sin of the angle between neighbouring sectors (O9)
    tpc_params p;
};

// One (task,row) bin after K1: where its hits are and the uniform (y,z) grid laid over them.  32 bytes = one
// sector; the second half alone (base, n, ny, nz) serves the paths that only need the hit range.
struct __align__(16) BinDesc {
    float y0, z0, idy, idz;   // cell = (int)((y - y0) * idy), (int)((z - z0) * idz), clamped
    int32_t base, n, ny, nz;  // first sorted hit (batch-global), hits, grid dims
};

// Everything a kernel may touch, for one batch.
struct SeedRec;
struct UpRec;

struct View {
    int32_t n_events, n_tasks, n_bins, N;
    const EventSrc* ev;      // [n_events]
    const int32_t* sec_off;  // [n_events][n_sectors+1] event-local
    // K1: bucket by (task,row), sort by grid cell
    int32_t* bin_count;      // [n_bins+1]
    int32_t* bin_start;      // [n_bins+1] exclusive scan of bin_count
    uint16_t* slot;          // [N] position of a cluster inside its bin, arrival order (batch-global cluster order)
    float4* thit;            // [N] bucketed, unsorted: (y, z, caller's index, -) -- one 16-byte record per scattered store
    int32_t* tidx;           // [N] scratch: K3's list of the start hits of each bin
    float2* shit; int32_t* sorig;  // [N] sorted by (task,row,cell): (y,z), caller's index in its event
    BinDesc* desc;           // [n_bins]
    uint16_t* cells;         // [kCellsPerHit*N + n_bins*kCellPad] first hit of each cell, relative to the bin's base
    // K2-K4
    int32_t *link_up, *link_dn, *clink_up, *clink_dn; // [N] batch-global sorted index or -1
    int32_t* seed_count;     // [n_bins+1]
    int32_t* seed_start;     // [n_bins+1]
    int32_t* seeds;          // [S_cap] sorted index of the start hit, canonical order
    int32_t* seed_bin;       // [S_cap]
    int32_t S_cap;
    // K5
    uint16_t* tl_tab;        // [S_cap][tab_stride] row -> row-local hit or kNoHit; valid for first_row..last_row
    int32_t tab_stride;
    int32_t* tl_rows;        // [S_cap] first_row | last_row << 8 | n_hits << 16
    float* tl_par;           // [6][S_cap] y z s t q chi2
    SeedRec* seed_rec;       // [S_cap] start hit and its up-link: coordinates and sorted indices (K4 -> K5 up sweep)
    UpRec* tl_up;            // [S_cap] what the up pass hands to the down pass, by tracklet
    UpRec* dn_rec;           // [S_cap] the same records, per task ordered by top row (written at the turn of the sweeps)
    uint32_t* kf_park;       // [S_cap] K5 scratch: per task, parked tracklets in order of parking (id in task | top row << 24)
    int32_t *dn_count, *dn_start, *dn_fill;   // [n_bins+1] O9: refitted tracks per (task, first fitted row)
    // K6
    uint32_t* owner;         // [N] best key among tracklets holding the hit
    int32_t* tl_nown;        // [S_cap+1] hits owned (0 when the track is dropped)
    int32_t* tl_keep;        // [S_cap+1] 1 when the track is kept
    int32_t* tl_cnt;         // [sel_C][S_cap] hits owned in each chunk of the task's pad rows
    int32_t sel_C;           // chunks per sector task in the selector
    int32_t* trk_scan;       // [S_cap+1]
    int32_t* hit_scan;       // [S_cap+1]
    int32_t* ev_off;         // [2][n_events+1] track / hit offsets of each event
    // outputs
    int32_t *o_sector, *o_first_hit, *o_n_hits, *o_ndf, *o_hit_idx;
    float *o_x, *o_y, *o_z, *o_sinphi, *o_tgl, *o_qpt, *o_chi2;
    // refit of the output tracks (tpc_params.refit): the tracks' hits as (y,z) and pad row, in hit-list order
    float2* o_hit_yz; uint8_t* o_hit_row;   // [N]
    int32_t* trk_hit0;       // [S_cap] first entry of a track's hit list in the batch's hit arrays
    int32_t* trk_rows;       // [S_cap] refit: reference row | outer row << 8, or -1 (no refit)
    int32_t* trk_task;       // [S_cap] sector task of a track (O9)
    float *o_xo, *o_yo, *o_zo, *o_so, *o_to, *o_qo;   // [S_cap] outer state of the refit (up pass at its top hit)
    int32_t *o_next, *o_prev;   // [S_cap] O9 links, event-local track index or -1
    int32_t* o_global;          // [S_cap] first segment of the chain a track belongs to, event-local
    // O10: fit of the global track, at its first segment
    float *o_gx, *o_gy, *o_gz, *o_gs, *o_gt, *o_gq, *o_gchi2;
    int32_t *o_gndf, *o_gnhits, *o_gsector;
    unsigned long long* cnt; // [CNT_N]
    unsigned long long* kf_cursor;  // [kNCursors] units of work handed out: [0] K5 sector tasks, [2] refit
};

__device__ __forceinline__ int lane_id() { return threadIdx.x & 31; }
__device__ __forceinline__ unsigned lanemask_lt() { return (1u << lane_id()) - 1u; }

__device__ __forceinline__ int4 load_desc_n(const View& v, int bin) {   // base, n, ny, nz
    return __ldg(reinterpret_cast<const int4*>(&v.desc[bin]) + 1);
}
__device__ __forceinline__ float4 load_desc_f(const View& v, int bin) { // y0, z0, idy, idz
    return __ldg(reinterpret_cast<const float4*>(&v.desc[bin]));
}
__device__ __forceinline__ const uint16_t* cell_table(const View& v, int bin, int base) {
    return v.cells + (size_t)kCellsPerHit * base + (size_t)bin * kCellPad;
}

__device__ __forceinline__ int grid_cell(float v, float v0, float iv, int n) {
    const int i = (int)((v - v0) * iv);
    return max(0, min(i, n - 1));
}

// Cell window of [y-wy, y+wy] x [z-wz, z+wz] (padded) in the grid (gf, ny, nz): columns iy0..iy1, rows iz0..iz1.
// A grid row's candidates are the contiguous hits cs[iz*ny+iy0] .. cs[iz*ny+iy1+1]; exact tests are the caller's.
struct CellWin { int iy0, iy1, iz0, iz1; };
__device__ __forceinline__ CellWin cell_window(const float4& gf, int ny, int nz, float y, float z, float wy, float wz) {
    CellWin w;
    w.iy0 = grid_cell(y - wy - kGridPad, gf.x, gf.z, ny); w.iy1 = grid_cell(y + wy + kGridPad, gf.x, gf.z, ny);
    w.iz0 = grid_cell(z - wz - kGridPad, gf.y, gf.w, nz); w.iz1 = grid_cell(z + wz + kGridPad, gf.y, gf.w, nz);
    return w;
}

}  // namespace tpc
