// sel_kernels.cuh -- K6 tracklet selector with the hit-ownership words of a sector task held in shared memory.
//
// owner[hit] = max key over the tracklets (n_hits >= min_tracklet_hits) holding the hit, key = n_hits << 24 |
// (2^24 - 1 - id within the task): more hits first, then the lower canonical id.  All tracklets
// that can hold a hit of sector task T belong to T, so the claims of a task touch only the task's own hits: a CTA
// takes one task -- or, when the task's hits do not fit the shared memory, one of C runs of consecutive pad rows
// of it ("chunk", balanced by hits) -- keeps the owner words of those hits in shared memory, and walks the
// task's tracklets twice: atomicMax of the keys, then the count of the hits each tracklet owns.  The random
// 4-byte gathers and atomics of the selection never leave the SM; global memory sees the row -> hit tables
// (read coalesced, one warp per tracklet) and one coalesced copy of the owner words.
#pragma once
#include "common.cuh"
#include "kf_kernels.cuh"

namespace tpc {

constexpr int kSelCtaThreads = 512;
constexpr int kSelCap = 26000;          // owner words of a chunk (104 KB: two CTAs per SM)
constexpr int kSelTile = 2048;          // tracklets whose kept members are listed at a time

// rows [r_lo, r_hi) of chunk c of task `tb / nr`: the rows whose first hit falls into the c-th of C equal
// shares of the task's hits.  s_base[r - r_lo] = first hit of row r (batch-global), one entry more than rows.
__device__ __forceinline__ void sel_chunk(const View& v, int tb, int nr, int c, int C, int& r_lo, int& r_hi) {
    const int b0 = v.bin_start[tb];
    const long long nt = v.bin_start[tb + nr] - b0;
    const int lo_hit = b0 + (int)(nt * c / C), hi_hit = b0 + (int)(nt * (c + 1) / C);
    // first row whose first hit is >= x (rows are in hit order; empty rows share their successor's first hit)
    auto first_row_at = [&](int x) {
        int lo = 0, hi = nr;
        while (lo < hi) {
            const int mid = (lo + hi) >> 1;
            if (v.bin_start[tb + mid] >= x) hi = mid; else lo = mid + 1;
        }
        return lo;
    };
    r_lo = c == 0 ? 0 : first_row_at(lo_hit);
    r_hi = c == C - 1 ? nr : first_row_at(hi_hit);
}

// K6a + K6b: claims and owned-hit counts of one (task, chunk); the owner words go back to global memory for K6c
__global__ void __launch_bounds__(kSelCtaThreads, 2) k_select_claim(const View v, const __grid_constant__ Const c) {
    extern __shared__ uint32_t s_owner[];
    __shared__ int32_t s_base[TPC_MAX_ROWS + 2];
    __shared__ uint16_t s_list[kSelTile];   // the tracklets of a tile that take part (offsets into the tile)
    __shared__ int32_t s_n;
    __shared__ unsigned long long s_claimed;
    TPC_RETURN_IF_REJECTED(v);
    const int C = v.sel_C, nr = c.n_rows;
    const int task = blockIdx.x / C, ch = blockIdx.x - task * C, tb = task * nr;
    const int lane = lane_id();
    int r_lo, r_hi;
    sel_chunk(v, tb, nr, ch, C, r_lo, r_hi);
    for (int r = r_lo + threadIdx.x; r <= r_hi; r += kSelCtaThreads) s_base[r - r_lo] = v.bin_start[tb + r];
    if (threadIdx.x == 0) s_claimed = 0ull;
    __syncthreads();
    const int h_lo = s_base[0], n_h = s_base[r_hi - r_lo] - h_lo;
    if (n_h > kSelCap) {   // the host sizes C so that this cannot happen
        if (threadIdx.x == 0) atomicOr((unsigned int*)&v.cnt[CNT_ERR], kErrSelCapacity);
        return;
    }
    for (int k = threadIdx.x; k < n_h; k += kSelCtaThreads) s_owner[k] = 0u;
    __syncthreads();
    const int S = min(v.seed_start[v.n_bins], v.S_cap);
    const int i0 = min(v.seed_start[tb], S), i1 = min(v.seed_start[tb + nr], S);
    // The task's row -> hit tables are one contiguous block; a thread takes 8 consecutive rows of one tracklet
    // (one 16-byte load), so the block streams through with every load independent of the others.
    const int g_lo = r_lo >> 3, G = max(((r_hi - 1) >> 3) - g_lo + 1, 1);   // (an empty chunk has r_hi == r_lo)
    unsigned claimed = 0;
    // The tracklets that take part (with the seed de-duplication two start hits in three build none) are listed
    // first, kSelTile start hits at a time, so that the lanes of the two passes are all at work.
    for (int pass = 0; pass < 2; pass++) {
        for (int tile = i0; tile < i1; tile += kSelTile) {
            __syncthreads();
            if (threadIdx.x == 0) s_n = 0;
            __syncthreads();
            for (int k = threadIdx.x; k < kSelTile; k += kSelCtaThreads) {
                const int i = tile + k;
                bool live = false;
                if (i < i1) {
                    const int pk = v.tl_rows[i];
                    live = (pk >> 16) >= c.p.min_tracklet_hits && max(pk & 0xff, r_lo) <= min((pk >> 8) & 0xff, r_hi - 1);
                }
                const unsigned m = __ballot_sync(kFull, live);
                int base = 0;
                if (lane == 0 && m) base = atomicAdd(&s_n, __popc(m));
                base = __shfl_sync(kFull, base, 0);
                if (live) s_list[base + __popc(m & lanemask_lt())] = (uint16_t)k;
            }
            __syncthreads();
            const int n_units = s_n * G;
            for (int u = threadIdx.x; u < n_units; u += kSelCtaThreads) {
                const int q = u / G, g = g_lo + (u - q * G);
                const int i = tile + (int)s_list[q], pk = v.tl_rows[i];
                const int nh = pk >> 16;
                const int a = max(pk & 0xff, r_lo), b = min((pk >> 8) & 0xff, r_hi - 1);
                const int r8 = g << 3;
                if (r8 > b || r8 + 7 < a) continue;
                const uint32_t key = ((uint32_t)nh << 24) | (uint32_t)(0xffffff - (i - i0));
                const uint4 qw = *reinterpret_cast<const uint4*>(v.tl_tab + (size_t)i * v.tab_stride + r8);
                const uint32_t w[4] = {qw.x, qw.y, qw.z, qw.w};
                int own = 0;
#pragma unroll
                for (int k = 0; k < 8; k++) {
                    const uint32_t e = (w[k >> 1] >> ((k & 1) * 16)) & 0xffffu;
                    const int r = r8 + k;
                    if (e != kNoHit && r >= a && r <= b) {
                        uint32_t* o = &s_owner[s_base[r - r_lo] - h_lo + (int)e];
                        if (pass == 0) { atomicMax(o, key); claimed++; }
                        else own += (*o == key);
                    }
                }
                if (pass == 1 && own) atomicAdd(&v.tl_cnt[(size_t)ch * v.S_cap + i], own);
            }
        }
        __syncthreads();
    }
    for (int k = threadIdx.x; k < n_h; k += kSelCtaThreads) v.owner[h_lo + k] = s_owner[k];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) claimed += __shfl_xor_sync(kFull, claimed, o);
    if (lane == 0 && claimed) atomicAdd(&s_claimed, (unsigned long long)claimed);
    __syncthreads();
    if (threadIdx.x == 0 && s_claimed) atomicAdd(&v.cnt[CNT_TL_HITS], s_claimed);
}

// a track is kept when its tracklet owns at least min_track_hits hits; entries beyond the start-hit count read 0
__global__ void __launch_bounds__(256) k_select_keep(const View v, int min_track_hits) {
    const int i = blockIdx.x * 256 + threadIdx.x;
    if (i > v.S_cap) return;
    const int S = min(v.seed_start[v.n_bins], v.S_cap);
    int own = 0;
    if (i < S)
        for (int ch = 0; ch < v.sel_C; ch++) own += v.tl_cnt[(size_t)ch * v.S_cap + i];
    const int keep = own >= min_track_hits;
    v.tl_keep[i] = keep;
    v.tl_nown[i] = keep ? own : 0;
}

// K6c: output tracks in canonical order; hit lists row-ascending.  The chunks of a task write the pieces of a
// hit list side by side: a chunk's piece starts behind the hits the lower chunks own.
__global__ void __launch_bounds__(kSelCtaThreads, 2) k_select_write(const View v, const __grid_constant__ Const c) {
    extern __shared__ uint32_t s_owner[];
    __shared__ int32_t s_base[TPC_MAX_ROWS + 2];
    __shared__ int32_t s_list[kSelTile];
    __shared__ int32_t s_n;
    TPC_RETURN_IF_REJECTED(v);
    const int C = v.sel_C, nr = c.n_rows;
    const int task = blockIdx.x / C, ch = blockIdx.x - task * C, tb = task * nr;
    const int lane = lane_id(), warp = threadIdx.x >> 5, n_warps = kSelCtaThreads / 32;
    int r_lo, r_hi;
    sel_chunk(v, tb, nr, ch, C, r_lo, r_hi);
    for (int r = r_lo + threadIdx.x; r <= r_hi; r += kSelCtaThreads) s_base[r - r_lo] = v.bin_start[tb + r];
    __syncthreads();
    const int h_lo = s_base[0], n_h = s_base[r_hi - r_lo] - h_lo;
    if (n_h > kSelCap) return;
    for (int k = threadIdx.x; k < n_h; k += kSelCtaThreads) s_owner[k] = v.owner[h_lo + k];
    __syncthreads();
    const int S = min(v.seed_start[v.n_bins], v.S_cap);
    const int i0 = min(v.seed_start[tb], S), i1 = min(v.seed_start[tb + nr], S);
    const int e = task / c.n_sectors;
    // A lane takes 8 consecutive rows of one kept tracklet (one 16-byte load); the G row groups of a tracklet sit
    // in G neighbouring lanes, so a warp works on 32 / G tracklets at once and a segmented scan over the groups'
    // owned-hit counts gives every group its place in the track's hit list.
    const int g_lo = r_lo >> 3, G = max(((r_hi - 1) >> 3) - g_lo + 1, 1);   // (an empty chunk has r_hi == r_lo)   // G <= 32
    const int T = 32 / G;
    const int tl = lane / G, gi = lane - tl * G, g = g_lo + gi;
    for (int tile = i0; tile < i1; tile += kSelTile) {
        __syncthreads();
        if (threadIdx.x == 0) s_n = 0;
        __syncthreads();
        for (int k = threadIdx.x; k < kSelTile; k += kSelCtaThreads) {   // the kept tracklets of the tile
            const int i = tile + k;
            const bool keep = i < i1 && v.tl_keep[i] != 0;
            const unsigned m = __ballot_sync(kFull, keep);
            int base = 0;
            if (lane == 0 && m) base = atomicAdd(&s_n, __popc(m));
            base = __shfl_sync(kFull, base, 0);
            if (keep) s_list[base + __popc(m & lanemask_lt())] = i;
        }
        __syncthreads();
        const int n_kept = s_n;
        for (int t0 = warp * T; t0 < n_kept; t0 += n_warps * T) {
            const bool on = tl < T && t0 + tl < n_kept;
            int own = 0, ho = 0, a = 0, b = -1, r8 = g << 3;
            uint32_t key = 0;
            uint32_t w[4] = {0u, 0u, 0u, 0u};
            if (on) {
                const int i = s_list[t0 + tl];
                const int pk = v.tl_rows[i];
                const int nh = pk >> 16, first = pk & 0xff, last = (pk >> 8) & 0xff;
                key = ((uint32_t)nh << 24) | (uint32_t)(0xffffff - (i - i0));
                ho = v.hit_scan[i];
                if (ch == 0 && gi == 0) {
                    const int ti = v.trk_scan[i];
                    const int sc = v.S_cap;
                    v.o_sector[ti] = task - e * c.n_sectors;
                    if (c.p.refit) { v.trk_hit0[ti] = ho; v.trk_task[ti] = task; }
                    v.o_first_hit[ti] = ho - v.ev_off[v.n_events + 1 + e];
                    v.o_n_hits[ti] = v.tl_nown[i];
                    v.o_ndf[ti] = 2 * nh - 5;
                    v.o_x[ti] = c.row_x[first];
                    v.o_y[ti] = v.tl_par[i]; v.o_z[ti] = v.tl_par[sc + i]; v.o_sinphi[ti] = v.tl_par[2 * sc + i];
                    v.o_tgl[ti] = v.tl_par[3 * sc + i]; v.o_qpt[ti] = v.tl_par[4 * sc + i]; v.o_chi2[ti] = v.tl_par[5 * sc + i];
                }
                for (int k = 0; k < ch; k++) ho += v.tl_cnt[(size_t)k * v.S_cap + i];
                a = max(first, r_lo); b = min(last, r_hi - 1);
                if (r8 <= b && r8 + 7 >= a) {
                    const uint4 q = *reinterpret_cast<const uint4*>(v.tl_tab + (size_t)i * v.tab_stride + r8);
                    w[0] = q.x; w[1] = q.y; w[2] = q.z; w[3] = q.w;
                } else b = -1;
            }
            int hits[8];
#pragma unroll
            for (int k = 0; k < 8; k++) {
                const uint32_t en = (w[k >> 1] >> ((k & 1) * 16)) & 0xffffu;
                const int r = r8 + k;
                int h = -1;
                if (r >= a && r <= b && en != kNoHit) {
                    h = s_base[r - r_lo] + (int)en;
                    if (s_owner[h - h_lo] != key) h = -1;
                }
                hits[k] = h;
                own += h >= 0;
            }
            int incl = own;   // scan over the G lanes of the tracklet
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { const int x = __shfl_up_sync(kFull, incl, o); if (gi >= o) incl += x; }
            int pos = ho + incl - own;
#pragma unroll
            for (int k = 0; k < 8; k++)
                if (hits[k] >= 0) {
                    v.o_hit_idx[pos] = v.sorig[hits[k]];
                    if (c.p.refit) { v.o_hit_yz[pos] = v.shit[hits[k]]; v.o_hit_row[pos] = (uint8_t)(r8 + k); }   // for O8
                    pos++;
                }
        }
    }
}

}  // namespace tpc
