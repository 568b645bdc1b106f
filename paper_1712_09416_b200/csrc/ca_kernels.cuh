// ca_kernels.cuh -- K1 (bucket + per-row grid sort), K2 (neighbour finder), K3 (cleaner), K4 (start hits).
// The arithmetic that decides a link is written exactly as DESIGN.md "O2" parenthesises it and compiled
// without contraction (-fmad=false), so that it rounds like the strict-float32 reference.
#pragma once
#include "common.cuh"
#include "scan.cuh"

namespace tpc {

// ---------------------------------------------------------------------------------------------------------
// K1a: count clusters per (task,row) bin; remember each cluster's arrival slot inside its bin.
// grid (ceil(max n / 256), n_events)
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ int sector_of(const int32_t* so, int ns, int i) {
    int lo = 0, hi = ns;  // largest s with so[s] <= i
    while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (so[mid] <= i) lo = mid; else hi = mid;
    }
    return lo;
}

constexpr int kCountPer = 8;                    // clusters per thread
constexpr int kCountChunk = 256 * kCountPer;    // clusters per CTA
constexpr int kCountBins = 2048;                // (sector,row) bins of a chunk counted in shared memory

__global__ void __launch_bounds__(256) k_count(const View v, const __grid_constant__ Const c, int ns, int nr) {
    __shared__ int32_t so[64 + 1];
    __shared__ int32_t hist[kCountBins];   // clusters of this chunk per bin, then the chunk's first slot in the bin
    const int e = blockIdx.y;
    const EventSrc src = v.ev[e];
    const int i0 = blockIdx.x * kCountChunk;
    if (i0 >= src.n) return;
    const int i1 = min(i0 + kCountChunk, src.n);
    for (int k = threadIdx.x; k <= ns; k += 256) so[k] = v.sec_off[e * (ns + 1) + k];
    __syncthreads();
    // a chunk of consecutive clusters spans few sectors: its bins are counted in shared memory and every bin
    // is then reserved with ONE global atomic per chunk
    const int s_lo = sector_of(so, ns, i0), s_hi = sector_of(so, ns, i1 - 1);
    const int nb = (s_hi - s_lo + 1) * nr;
    const int bin0 = (e * ns + s_lo) * nr;
    const bool local = nb <= kCountBins;
    if (local) for (int b = threadIdx.x; b < nb; b += 256) hist[b] = 0;
    __syncthreads();
    uint32_t pk[kCountPer];   // bin within the chunk << 12 | arrival rank within the chunk
#pragma unroll
    for (int k = 0; k < kCountPer; k++) {
        const int i = i0 + k * 256 + threadIdx.x;
        pk[k] = 0xffffffffu;
        if (i < i1) {
            const int r = src.row[i];
            if (r < 0 || r >= nr) { atomicOr((unsigned int*)&v.cnt[CNT_ERR], kErrBadRow); continue; }
            if (c.p.checked) {   // S23: coordinates finite, x on its pad row
                const float yy = src.y[i], zz = src.z[i];
                bool bad = !(fabsf(yy) <= 3.0e38f) || !(fabsf(zz) <= 3.0e38f);
                if (src.x) bad = bad || !(fabsf(src.x[i] - c.row_x[r]) <= 1.0e-3f);
                if (bad) atomicOr((unsigned int*)&v.cnt[CNT_ERR], kErrBadInput);
            }
            int s = s_lo;
            while (i >= so[s + 1]) s++;
            const int bl = (s - s_lo) * nr + r;
            if (local) pk[k] = ((uint32_t)bl << 12) | (uint32_t)atomicAdd(&hist[bl], 1);
            else {
                const int sl = atomicAdd(&v.bin_count[bin0 + bl], 1);
                if (sl >= TPC_MAX_ROW_HITS) atomicOr((unsigned int*)&v.cnt[CNT_ERR], kErrRowCapacity);
                v.slot[src.off + i] = (uint16_t)min(sl, 65535);
            }
        }
    }
    if (!local) return;
    __syncthreads();
    for (int b = threadIdx.x; b < nb; b += 256) {
        const int cnt = hist[b];
        if (cnt) hist[b] = atomicAdd(&v.bin_count[bin0 + b], cnt);
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < kCountPer; k++) {
        if (pk[k] == 0xffffffffu) continue;
        const int i = i0 + k * 256 + threadIdx.x;
        const int sl = hist[pk[k] >> 12] + (int)(pk[k] & 0xfffu);
        if (sl >= TPC_MAX_ROW_HITS) atomicOr((unsigned int*)&v.cnt[CNT_ERR], kErrRowCapacity);
        v.slot[src.off + i] = (uint16_t)min(sl, 65535);
    }
}

// K1b: move (y, z, index) into the bin, arrival order.  kScatterPer clusters per thread, all loads of a thread
// issued before the first dependent one (the kernel waits on memory latency, not on bandwidth).
constexpr int kScatterPer = 4;
constexpr int kScatterChunk = 256 * kScatterPer;

__global__ void __launch_bounds__(256) k_scatter(const View v, int ns, int nr) {
    __shared__ int32_t so[64 + 1];
    const int e = blockIdx.y;
    const EventSrc src = v.ev[e];
    const int i0 = blockIdx.x * kScatterChunk;
    if (i0 >= src.n) return;
    for (int k = threadIdx.x; k <= ns; k += 256) so[k] = v.sec_off[e * (ns + 1) + k];
    int r[kScatterPer], sl[kScatterPer];
    float2 h[kScatterPer];
#pragma unroll
    for (int j = 0; j < kScatterPer; j++) {
        const int i = i0 + j * 256 + threadIdx.x;
        r[j] = -1; sl[j] = 0; h[j] = make_float2(0.f, 0.f);
        if (i < src.n) {
            r[j] = src.row[i]; sl[j] = v.slot[src.off + i];
            h[j] = make_float2(src.y[i], src.z[i]);
        }
    }
    __syncthreads();
    int pos[kScatterPer];
#pragma unroll
    for (int j = 0; j < kScatterPer; j++) {
        const int i = i0 + j * 256 + threadIdx.x;
        pos[j] = -1;
        if (r[j] >= 0 && r[j] < nr && sl[j] < TPC_MAX_ROW_HITS)
            pos[j] = __ldg(&v.bin_start[(e * ns + sector_of(so, ns, i)) * nr + r[j]]) + sl[j];
    }
#pragma unroll
    for (int j = 0; j < kScatterPer; j++)
        if (pos[j] >= 0) v.thit[pos[j]] = make_float4(h[j].x, h[j].y, __int_as_float(i0 + j * 256 + (int)threadIdx.x), 0.f);   // one 16-byte store
}

// ---------------------------------------------------------------------------------------------------------
// K1c: one CTA per bin: bounding box -> grid dims -> counting sort of the bin by grid cell -> cell table.
// The grid only accelerates the window searches; windows are defined on coordinates and every tie is broken
// on the caller's index, so neither the grid's shape nor the order inside a cell changes a result.
// A bin of up to kSortReg * kSortThreads hits (every pad row of a central event) is read ONCE, into registers.
// ---------------------------------------------------------------------------------------------------------
#ifndef TPC_SORT_THREADS
#define TPC_SORT_THREADS 128
#endif
constexpr int kSortThreads = TPC_SORT_THREADS;
constexpr int kSortReg = 4;

// SMALL: the bins of up to kSortReg * kSortThreads hits (little shared memory: many CTAs per SM); the other launch
// takes the larger ones
#ifndef TPC_SORT_BLOCKS
#define TPC_SORT_BLOCKS 12
#endif
template <bool SMALL>
__global__ void __launch_bounds__(kSortThreads, SMALL ? TPC_SORT_BLOCKS : 7) k_sort_row(const View v) {
    constexpr int kCells = SMALL ? kCellsPerHit * kSortReg * kSortThreads + kCellPad : kMaxCells;
    __shared__ int cnt[kCells + 1];                                   // hits per cell, then first hit of each cell
    __shared__ uint16_t ck[SMALL ? 1 : TPC_MAX_ROW_HITS];             // cell of hit k
    __shared__ uint16_t rk[SMALL ? 1 : TPC_MAX_ROW_HITS];             // arrival rank of hit k inside its cell
    __shared__ float red[4][kSortThreads / 32];
    __shared__ int scan_total;
    // SMALL: a CTA per bin, the larger bins are listed (in seed_count, free until K3); the other launch is a fixed
    // grid that takes the listed bins in turn
    for (int bi = blockIdx.x; SMALL ? bi == (int)blockIdx.x : bi < (int)v.cnt[CNT_LARGE_BINS]; bi += gridDim.x) {
    const int bin = SMALL ? bi : v.seed_count[bi];
    const int b0 = v.bin_start[bin];
    const int n = min(v.bin_start[bin + 1] - b0, TPC_MAX_ROW_HITS);
    if (SMALL && n > kSortReg * kSortThreads) {
        if (threadIdx.x == 0) v.seed_count[(int)atomicAdd(&v.cnt[CNT_LARGE_BINS], 1ull)] = bin;
        return;
    }
    if (!SMALL) __syncthreads();   // the shared arrays are free again
    uint16_t* cs = v.cells + (size_t)kCellsPerHit * b0 + (size_t)bin * kCellPad;
    if (n == 0) {
        if (threadIdx.x == 0) {
            BinDesc d; d.y0 = 0.f; d.z0 = 0.f; d.idy = 0.f; d.idz = 0.f; d.base = b0; d.n = 0; d.ny = 1; d.nz = 1;
            v.desc[bin] = d;
            cs[0] = 0; cs[1] = 0;
        }
        return;
    }
    constexpr bool small = SMALL;
    float2 hr[kSortReg];
    int ir[kSortReg];
    // bounding box
    float ymin = 3.0e38f, ymax = -3.0e38f, zmin = 3.0e38f, zmax = -3.0e38f;
    if (small) {
#pragma unroll
        for (int j = 0; j < kSortReg; j++) {
            const int k = j * kSortThreads + threadIdx.x;
            if (k < n) { const float4 q = v.thit[b0 + k]; hr[j] = make_float2(q.x, q.y); ir[j] = __float_as_int(q.z); }
        }
#pragma unroll
        for (int j = 0; j < kSortReg; j++)
            if (j * kSortThreads + (int)threadIdx.x < n) {
                ymin = fminf(ymin, hr[j].x); ymax = fmaxf(ymax, hr[j].x); zmin = fminf(zmin, hr[j].y); zmax = fmaxf(zmax, hr[j].y);
            }
    } else {
        for (int k = threadIdx.x; k < n; k += kSortThreads) {
            const float4 h = v.thit[b0 + k];
            ymin = fminf(ymin, h.x); ymax = fmaxf(ymax, h.x); zmin = fminf(zmin, h.y); zmax = fmaxf(zmax, h.y);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        ymin = fminf(ymin, __shfl_xor_sync(kFull, ymin, o)); ymax = fmaxf(ymax, __shfl_xor_sync(kFull, ymax, o));
        zmin = fminf(zmin, __shfl_xor_sync(kFull, zmin, o)); zmax = fmaxf(zmax, __shfl_xor_sync(kFull, zmax, o));
    }
    if (lane_id() == 0) {
        const int w = threadIdx.x >> 5;
        red[0][w] = ymin; red[1][w] = ymax; red[2][w] = zmin; red[3][w] = zmax;
    }
    __syncthreads();
#pragma unroll
    for (int w = 0; w < kSortThreads / 32; w++) {   // min / max: the same value in every thread, whatever the order
        ymin = fminf(ymin, red[0][w]); ymax = fmaxf(ymax, red[1][w]);
        zmin = fminf(zmin, red[2][w]); zmax = fmaxf(zmax, red[3][w]);
    }
    // grid dims: cells of about one hit's area, ~0.6 : 1/0.6 in (y : z), then kCellsPerHit times finer in y (the
    // hits of the cells iy0..iy1 of one grid row are contiguous, so fine y cells cost no extra range), never finer
    // than 0.35 x 1.2 cm
    const float ylen = fmaxf(ymax - ymin, 1.0e-3f), zlen = fmaxf(zmax - zmin, 1.0e-3f);
    const float area = ylen * zlen / (float)n;
    const float dy = fmaxf(sqrtf(area * 0.6f) / (float)kCellsPerHit, 0.35f), dz = fmaxf(sqrtf(area / 0.6f), 1.2f);
    int nz = max(1, min((int)(zlen / dz) + 1, 255));
    int ny = max(1, min((int)(ylen / dy) + 1, 255));
    const int cap = min(kCellsPerHit * n + kCellPad - 1, kMaxCells);  // ny*nz + 1 entries must fit
    if (nz > cap) nz = cap;
    if (ny * nz > cap) ny = max(1, cap / nz);
    const float idy = (float)ny / (ylen * 1.0001f), idz = (float)nz / (zlen * 1.0001f);
    const int ncell = ny * nz;
    for (int q = threadIdx.x; q <= ncell; q += kSortThreads) cnt[q] = 0;
    __syncthreads();
    int ckr[kSortReg], rkr[kSortReg];
    if (small) {
#pragma unroll
        for (int j = 0; j < kSortReg; j++)
            if (j * kSortThreads + (int)threadIdx.x < n) {
                ckr[j] = grid_cell(hr[j].y, zmin, idz, nz) * ny + grid_cell(hr[j].x, ymin, idy, ny);
                rkr[j] = atomicAdd(&cnt[ckr[j]], 1);
            }
    } else {
        for (int k = threadIdx.x; k < n; k += kSortThreads) {
            const float4 h = v.thit[b0 + k];
            const int cell = grid_cell(h.y, zmin, idz, nz) * ny + grid_cell(h.x, ymin, idy, ny);
            ck[k] = (uint16_t)cell;
            rk[k] = (uint16_t)atomicAdd(&cnt[cell], 1);
        }
    }
    __syncthreads();
    // exclusive scan of cnt[0..ncell): each thread owns a contiguous chunk
    {
        const int per = (ncell + kSortThreads - 1) / kSortThreads;
        const int q0 = threadIdx.x * per, q1 = min(q0 + per, ncell);
        int s = 0;
        for (int q = q0; q < q1; q++) s += cnt[q];
        int ex = block_excl_scan<kSortThreads>(s, &scan_total);
        for (int q = q0; q < q1; q++) { const int t = cnt[q]; cnt[q] = ex; ex += t; }
    }
    __syncthreads();
    for (int q = threadIdx.x; q <= ncell; q += kSortThreads) cs[q] = (uint16_t)(q < ncell ? cnt[q] : n);
    if (small) {
#pragma unroll
        for (int j = 0; j < kSortReg; j++)
            if (j * kSortThreads + (int)threadIdx.x < n) {
                const int pos = b0 + cnt[ckr[j]] + rkr[j];
                v.shit[pos] = hr[j];
                v.sorig[pos] = ir[j];
            }
    } else {
        for (int k = threadIdx.x; k < n; k += kSortThreads) {
            const int pos = b0 + cnt[ck[k]] + rk[k];
            const float4 q = v.thit[b0 + k];
            v.shit[pos] = make_float2(q.x, q.y);
            v.sorig[pos] = __float_as_int(q.z);
        }
    }
    if (threadIdx.x == 0) {
        BinDesc d; d.y0 = ymin; d.z0 = zmin; d.idy = idy; d.idz = idz; d.base = b0; d.n = n; d.ny = ny; d.nz = nz;
        v.desc[bin] = d;
    }
    }
}

// ---------------------------------------------------------------------------------------------------------
// K2 neighbour finder.  One CTA per bin (task,row); the two neighbour rows (hits + cell tables)
// are staged in shared memory; a thread takes hits of the row.
// For hit h of row r: among up-candidates u (row r+D) and down-candidates d (row r-D) inside the windows,
// minimise D = (y0 - yhat)^2 + (z0 - zhat)^2 with (yhat, zhat) the point of the line d->u at x0;
// ties -> lowest caller's index of u, then of d.
// ---------------------------------------------------------------------------------------------------------
constexpr int kNfThreads = 128;
#ifndef TPC_NF_CAP
#define TPC_NF_CAP 448
#endif
#ifndef TPC_NF_BLOCKS
#define TPC_NF_BLOCKS 12
#endif
constexpr int kNfCap = TPC_NF_CAP;   // hits of a neighbour row held in shared memory; larger rows are read in place
constexpr int kNfList = 8;     // candidates of a window remembered per hit; more -> nested walk

__global__ void __launch_bounds__(kNfThreads, TPC_NF_BLOCKS) k_neighbours(const View v, const __grid_constant__ Const c) {
    __shared__ float2 s_hu[kNfCap], s_hd[kNfCap];
    constexpr int kNfCells = kCellsPerHit * kNfCap + kCellPad;   // cell-table entries held in shared memory
    __shared__ uint16_t s_cu[kNfCells], s_cd[kNfCells];
    __shared__ uint16_t s_dl[kNfList][kNfThreads], s_ul[kNfList][kNfThreads];   // row-local candidates of the thread's hit
    TPC_RETURN_IF_REJECTED(v);
    const int bin = blockIdx.x;
    const int nr = c.n_rows, D = c.p.link_step;
    const int r = bin % nr;
    const int4 own = load_desc_n(v, bin);
    const int b0 = own.x, n = own.y;
    if (n == 0) return;
    bool none = (r - D < 0 || r + D >= nr);
    int4 du = make_int4(0, 0, 1, 1), dd = du;
    if (!none) {
        du = load_desc_n(v, bin + D); dd = load_desc_n(v, bin - D);
        none = du.y == 0 || dd.y == 0;
    }
    if (none) {
        for (int k = threadIdx.x; k < n; k += kNfThreads) { v.link_up[b0 + k] = -1; v.link_dn[b0 + k] = -1; }
        return;
    }
    const float4 gfu = load_desc_f(v, bin + D), gfd = load_desc_f(v, bin - D);
    const float2* hu = v.shit + du.x; const float2* hd = v.shit + dd.x;
    const uint16_t* cu = cell_table(v, bin + D, du.x); const uint16_t* cd = cell_table(v, bin - D, dd.x);
    if (du.y <= kNfCap && du.z * du.w < kNfCells) {
        for (int k = threadIdx.x; k < du.y; k += kNfThreads) s_hu[k] = hu[k];
        for (int k = threadIdx.x; k <= du.z * du.w; k += kNfThreads) s_cu[k] = cu[k];
        hu = s_hu; cu = s_cu;
    }
    if (dd.y <= kNfCap && dd.z * dd.w < kNfCells) {
        for (int k = threadIdx.x; k < dd.y; k += kNfThreads) s_hd[k] = hd[k];
        for (int k = threadIdx.x; k <= dd.z * dd.w; k += kNfThreads) s_cd[k] = cd[k];
        hd = s_hd; cd = s_cd;
    }
    __syncthreads();
    // The common case -- both neighbour rows staged -- is compiled apart with the shared-memory arrays named directly:
    // the loads of the hot loops are then LDS with immediate offsets, not generic loads that find their space at run time
    auto all_hits = [&](const float2* hu, const float2* hd, const uint16_t* cu, const uint16_t* cd) __attribute__((always_inline)) {
    const float x0 = c.row_x[r], x1 = c.row_x[r + D], x2 = c.row_x[r - D];
    const float wyu = c.p.nf_slope_y * fabsf(x1 - x0) + c.p.nf_w0, wzu = c.p.nf_slope_z * fabsf(x1 - x0) + c.p.nf_w0;
    const float wyd = c.p.nf_slope_y * fabsf(x2 - x0) + c.p.nf_w0, wzd = c.p.nf_slope_z * fabsf(x2 - x0) + c.p.nf_w0;
    const float a = (x0 - x2) / (x1 - x2);
    const int nyu = du.z, nyd = dd.z;
    for (int k = threadIdx.x; k < n; k += kNfThreads) {
        const int h = b0 + k;
        const float2 h0 = v.shit[h];
        const float y0 = h0.x, z0 = h0.y;
        int bpair = -1;         // row-local indices of the best pair, u << 16 | d (both < 2048)
        float best = __int_as_float(0x7f800000);   // +inf: the first pair always wins
        auto eval = [&](int u, const float2& pu, int d, const float2& pd) {
            const float yh = pd.x + a * (pu.x - pd.x);
            const float zh = pd.y + a * (pu.y - pd.y);
            const float dy = y0 - yh, dz = z0 - zh;
            const float dev = dy * dy + dz * dz;
            bool take = dev < best;
            if (dev == best) {  // exact tie (dev is finite, so a pair is held): lowest caller's index of u, then of d
                const int bu = bpair >> 16, bd = bpair & 0xffff;
                const int ou = v.sorig[du.x + u], obu = v.sorig[du.x + bu];
                take = ou < obu || (ou == obu && v.sorig[dd.x + d] < v.sorig[dd.x + bd]);
            }
            if (take) { best = dev; bpair = (u << 16) | d; }
        };
        // The candidates inside the two windows are first collected -- up to kNfList of each side, row-local indices
        // in shared memory -- and the pairs are then evaluated in ONE flat loop: a warp's trip count is its largest
        // pair count, not the sum over nested loops with diverging trip counts.
        const CellWin wd = cell_window(gfd, nyd, dd.w, y0, z0, wyd, wzd);
        int nd = 0, nu = 0;
        for (int iz = wd.iz0; iz <= wd.iz1; iz++) {
            int p = cd[iz * nyd + wd.iy0];
            const int pe = cd[iz * nyd + wd.iy1 + 1];
            for (; p < pe; p++) {
                const float2 pd = hd[p];
                if (fabsf(pd.x - y0) <= wyd && fabsf(pd.y - z0) <= wzd) {
                    if (nd < kNfList) s_dl[nd][threadIdx.x] = (uint16_t)p;
                    nd++;
                }
            }
        }
        CellWin wu = wd;
        if (nd > 0) {
            wu = cell_window(gfu, nyu, du.w, y0, z0, wyu, wzu);
            for (int iz = wu.iz0; iz <= wu.iz1; iz++) {
                int p = cu[iz * nyu + wu.iy0];
                const int pe = cu[iz * nyu + wu.iy1 + 1];
                for (; p < pe; p++) {
                    const float2 pu = hu[p];
                    if (fabsf(pu.x - y0) <= wyu && fabsf(pu.y - z0) <= wzu) {
                        if (nu < kNfList) s_ul[nu][threadIdx.x] = (uint16_t)p;
                        nu++;
                    }
                }
            }
        }
        if (nd <= kNfList && nu <= kNfList) {
            const int np = nd * nu;
            int ju = 0, jd = 0;
            for (int q = 0; q < np; q++) {
                const int u = s_ul[ju][threadIdx.x], d = s_dl[jd][threadIdx.x];
                eval(u, hu[u], d, hd[d]);
                if (++jd == nd) { jd = 0; ju++; }
            }
        } else if (nu > 0) {   // a crowded window: walk both again, nested
            for (int iz = wu.iz0; iz <= wu.iz1; iz++) {
                int p = cu[iz * nyu + wu.iy0];
                const int pe = cu[iz * nyu + wu.iy1 + 1];
                for (; p < pe; p++) {
                    const float2 pu = hu[p];
                    if (!(fabsf(pu.x - y0) <= wyu && fabsf(pu.y - z0) <= wzu)) continue;
                    for (int jz = wd.iz0; jz <= wd.iz1; jz++) {
                        int q = cd[jz * nyd + wd.iy0];
                        const int qe = cd[jz * nyd + wd.iy1 + 1];
                        for (; q < qe; q++) {
                            const float2 pd = hd[q];
                            if (fabsf(pd.x - y0) <= wyd && fabsf(pd.y - z0) <= wzd) eval(p, pu, q, pd);
                        }
                    }
                }
            }
        }
        const bool ok = bpair >= 0 && best <= c.p.nf_dmax;
        v.link_up[h] = ok ? du.x + (bpair >> 16) : -1;
        v.link_dn[h] = ok ? dd.x + (bpair & 0xffff) : -1;
    }
    };
    if (hu == s_hu && hd == s_hd) all_hits(s_hu, s_hd, s_cu, s_cd);
    else all_hits(hu, hd, cu, cd);
}

// ---------------------------------------------------------------------------------------------------------
// K3 cleaner + start-hit count.  clink_up[h] = link_up[h] if link_dn[link_up[h]] == h, else -1 (and the
// mirror image); one simultaneous pass.  A start hit has a cleaned up-link and no cleaned down-link.
// ---------------------------------------------------------------------------------------------------------
constexpr int kCleanThreads = 128;

// CLEAN false (stage-isolated runs, tpc_debug_resume): the cleaned links are taken as they stand
template <bool CLEAN>
__global__ void __launch_bounds__(kCleanThreads) k_clean(const View v) {
    __shared__ int nstart, nlink;
    TPC_RETURN_IF_REJECTED(v);
    const int bin = blockIdx.x;
    const int b0 = v.bin_start[bin], n = v.bin_start[bin + 1] - b0;
    if (threadIdx.x == 0) { nstart = 0; nlink = 0; }
    __syncthreads();
    int nl = 0;
    for (int k0 = 0; k0 < n; k0 += kCleanThreads) {
        const int k = k0 + threadIdx.x;
        bool st = false;
        if (k < n) {
            const int h = b0 + k;
            int cu, cd;
            if (CLEAN) {
                const int u = v.link_up[h], d = v.link_dn[h];
                cu = (u >= 0 && v.link_dn[u] == h) ? u : -1;
                cd = (d >= 0 && v.link_up[d] == h) ? d : -1;
                v.clink_up[h] = cu;
                v.clink_dn[h] = cd;
            } else {
                cu = v.clink_up[h]; cd = v.clink_dn[h];
            }
            st = cu >= 0 && cd < 0;
            nl += (cu >= 0);
        }
        // the row's start hits, in any order, into the bin's stretch of the (now free) bucket index array: K4
        // then reads a short list instead of the row's links
        const unsigned m = __ballot_sync(kFull, st);
        int basep = 0;
        if (lane_id() == 0 && m) basep = atomicAdd(&nstart, __popc(m));
        basep = __shfl_sync(kFull, basep, 0);
        if (st) v.tidx[b0 + basep + __popc(m & lanemask_lt())] = b0 + k;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) nl += __shfl_xor_sync(kFull, nl, o);
    if (lane_id() == 0 && nl) atomicAdd(&nlink, nl);
    __syncthreads();
    if (threadIdx.x == 0) {
        v.seed_count[bin] = nstart;
        if (nlink) atomicAdd(&v.cnt[CNT_LINKS], (unsigned long long)nlink);
    }
}

// ---------------------------------------------------------------------------------------------------------
// K4 start-hit compaction in canonical order (task, row, caller's index): K3 collected the row's start hits with
// warp ballots + prefix popcounts; here a rank by caller's index orders them.
// ---------------------------------------------------------------------------------------------------------
constexpr int kSeedThreads = 256;
constexpr int kSeedWarps = kSeedThreads / 32;   // a warp per bin: no block barrier, eight bins per CTA
constexpr int kSeedList = 128;                  // start hits of a bin ranked by its warp; more (the lowest rows of a sector,
                                                // where every long track starts): by the whole CTA afterwards

// start hit number `rank` of bin `bin`: the canonical list and the record the up pass starts from
__device__ __forceinline__ void seed_write(const View& v, const Const& c, int bin, int s0, int rank, int h0) {
    if (s0 + rank >= v.S_cap) { atomicOr((unsigned int*)&v.cnt[CNT_ERR], kErrSeedCapacity); return; }
    const int h1 = v.clink_up[h0];
    v.seeds[s0 + rank] = h0; v.seed_bin[s0 + rank] = bin;
    const float2 a0 = v.shit[h0], a1 = v.shit[h1];
    // initial direction of the up pass: s = dy / dl, t = dz / dl along the first link
    const int r = bin % c.n_rows;
    const float dx = c.row_x[r + c.p.link_step] - c.row_x[r];
    const float dy = a1.x - a0.x, dz = a1.y - a0.y;
    const float dl = sqrtf(dx * dx + dy * dy);
    float4* rec = reinterpret_cast<float4*>(v.seed_rec) + 2 * (size_t)(s0 + rank);
    rec[0] = make_float4(a0.x, a0.y, dy / dl, dz / dl);
    rec[1] = make_float4(__int_as_float(h0), __int_as_float(h1), __int_as_float(v.clink_up[h1]), 0.f);
}

__global__ void __launch_bounds__(kSeedThreads) k_seeds(const View v, const __grid_constant__ Const c) {
    __shared__ int list_h[kSeedWarps][kSeedList];
    __shared__ int list_o[kSeedWarps][kSeedList];
    __shared__ int big_h[TPC_MAX_ROW_HITS], big_o[TPC_MAX_ROW_HITS];
    __shared__ int s_big[kSeedWarps];
    TPC_RETURN_IF_REJECTED(v);
    const int warp = threadIdx.x >> 5, lane = lane_id();
    {
        const int bin = blockIdx.x * kSeedWarps + warp;
        int ns = 0, s0 = 0;
        if (bin < v.n_bins) { s0 = v.seed_start[bin]; ns = v.seed_start[bin + 1] - s0; }
        if (lane == 0) s_big[warp] = ns > kSeedList;
        if (ns > 0 && ns <= kSeedList) {
            const int b0 = v.bin_start[bin];
            for (int i = lane; i < ns; i += 32) {   // the list K3 left (any order)
                const int h = v.tidx[b0 + i];
                list_h[warp][i] = h;
                list_o[warp][i] = v.sorig[h];
            }
            __syncwarp();
            for (int i = lane; i < ns; i += 32) {
                const int o = list_o[warp][i];
                int rank = 0;
                for (int j = 0; j < ns; j++) rank += (list_o[warp][j] < o);
                seed_write(v, c, bin, s0, rank, list_h[warp][i]);
            }
        }
    }
    __syncthreads();
    for (int w = 0; w < kSeedWarps; w++) {
        if (!s_big[w]) continue;   // (uniform)
        const int bin = blockIdx.x * kSeedWarps + w;
        const int s0 = v.seed_start[bin], ns = min(v.seed_start[bin + 1] - s0, TPC_MAX_ROW_HITS);
        const int b0 = v.bin_start[bin];
        __syncthreads();
        for (int i = threadIdx.x; i < ns; i += kSeedThreads) {
            const int h = v.tidx[b0 + i];
            big_h[i] = h;
            big_o[i] = v.sorig[h];
        }
        __syncthreads();
        for (int i = threadIdx.x; i < ns; i += kSeedThreads) {
            const int o = big_o[i];
            int rank = 0;
            for (int j = 0; j < ns; j++) rank += (big_o[j] < o);
            seed_write(v, c, bin, s0, rank, big_h[i]);
        }
    }
}

}  // namespace tpc
