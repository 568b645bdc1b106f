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

__global__ void __launch_bounds__(256) k_count(const View v, int ns, int nr) {
    __shared__ int32_t so[64 + 1];
    const int e = blockIdx.y;
    const EventSrc src = v.ev[e];
    if (blockIdx.x * 256 >= src.n) return;
    for (int k = threadIdx.x; k <= ns; k += 256) so[k] = v.sec_off[e * (ns + 1) + k];
    __syncthreads();
    const int i = blockIdx.x * 256 + threadIdx.x;
    if (i >= src.n) return;
    const int r = src.row[i];
    if (r < 0 || r >= nr) { atomicOr((unsigned int*)&v.cnt[CNT_ERR], kErrBadRow); return; }
    const int s = sector_of(so, ns, i);
    const int bin = (e * ns + s) * nr + r;
    const int sl = atomicAdd(&v.bin_count[bin], 1);
    if (sl >= TPC_MAX_ROW_HITS) atomicOr((unsigned int*)&v.cnt[CNT_ERR], kErrRowCapacity);
    v.slot[src.off + i] = (uint16_t)min(sl, 65535);
}

// K1b: move (y, z, index) into the bin, arrival order.
__global__ void __launch_bounds__(256) k_scatter(const View v, int ns, int nr) {
    __shared__ int32_t so[64 + 1];
    const int e = blockIdx.y;
    const EventSrc src = v.ev[e];
    if (blockIdx.x * 256 >= src.n) return;
    for (int k = threadIdx.x; k <= ns; k += 256) so[k] = v.sec_off[e * (ns + 1) + k];
    __syncthreads();
    const int i = blockIdx.x * 256 + threadIdx.x;
    if (i >= src.n) return;
    const int r = src.row[i];
    if (r < 0 || r >= nr) return;
    const int s = sector_of(so, ns, i);
    const int bin = (e * ns + s) * nr + r;
    const int sl = v.slot[src.off + i];
    if (sl >= TPC_MAX_ROW_HITS) return;
    const int pos = v.bin_start[bin] + sl;
    v.ty[pos] = src.y[i];
    v.tz[pos] = src.z[i];
    v.tidx[pos] = i;
}

// ---------------------------------------------------------------------------------------------------------
// K1c: one CTA per bin: bounding box -> grid dims -> sort the bin by (cell, caller's index) -> cell table.
// The grid only accelerates the window searches; windows are defined on coordinates, so its shape never
// changes a result.
// ---------------------------------------------------------------------------------------------------------
constexpr int kSortThreads = 256;

__global__ void __launch_bounds__(kSortThreads) k_sort_row(const View v) {
    __shared__ unsigned long long key[TPC_MAX_ROW_HITS];
    __shared__ float red[4][kSortThreads / 32];
    __shared__ float box[4];
    const int bin = blockIdx.x;
    const int b0 = v.bin_start[bin];
    const int n = min(v.bin_start[bin + 1] - b0, TPC_MAX_ROW_HITS);
    uint16_t* cs = v.cells + (size_t)b0 + (size_t)bin * kCellPad;
    if (n == 0) {
        if (threadIdx.x == 0) {
            v.grid_f[bin] = make_float4(0.f, 0.f, 0.f, 0.f);
            v.grid_n[bin] = make_int2(1, 1);
            cs[0] = 0; cs[1] = 0;
        }
        return;
    }
    // bounding box
    float ymin = 3.0e38f, ymax = -3.0e38f, zmin = 3.0e38f, zmax = -3.0e38f;
    for (int k = threadIdx.x; k < n; k += kSortThreads) {
        const float y = v.ty[b0 + k], z = v.tz[b0 + k];
        ymin = fminf(ymin, y); ymax = fmaxf(ymax, y); zmin = fminf(zmin, z); zmax = fmaxf(zmax, z);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        ymin = fminf(ymin, __shfl_xor_sync(0xffffffffu, ymin, o)); ymax = fmaxf(ymax, __shfl_xor_sync(0xffffffffu, ymax, o));
        zmin = fminf(zmin, __shfl_xor_sync(0xffffffffu, zmin, o)); zmax = fmaxf(zmax, __shfl_xor_sync(0xffffffffu, zmax, o));
    }
    if (lane_id() == 0) {
        const int w = threadIdx.x >> 5;
        red[0][w] = ymin; red[1][w] = ymax; red[2][w] = zmin; red[3][w] = zmax;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < kSortThreads / 32; w++) {
            ymin = fminf(ymin, red[0][w]); ymax = fmaxf(ymax, red[1][w]);
            zmin = fminf(zmin, red[2][w]); zmax = fmaxf(zmax, red[3][w]);
        }
        box[0] = ymin; box[1] = ymax; box[2] = zmin; box[3] = zmax;
    }
    __syncthreads();
    ymin = box[0]; ymax = box[1]; zmin = box[2]; zmax = box[3];
    // grid dims: about one cell per hit, cells ~0.6 : 1/0.6 in (y : z), never finer than 0.7 x 1.2 cm
    const float ylen = fmaxf(ymax - ymin, 1.0e-3f), zlen = fmaxf(zmax - zmin, 1.0e-3f);
    const float area = ylen * zlen / (float)n;
    const float dy = fmaxf(sqrtf(area * 0.6f), 0.7f), dz = fmaxf(sqrtf(area / 0.6f), 1.2f);
    int nz = max(1, min((int)(zlen / dz) + 1, 255));
    int ny = max(1, min((int)(ylen / dy) + 1, 255));
    const int cap = n + kCellPad - 1;  // ny*nz + 1 entries must fit
    if (nz > cap) nz = cap;
    if (ny * nz > cap) ny = max(1, cap / nz);
    const float idy = (float)ny / (ylen * 1.0001f), idz = (float)nz / (zlen * 1.0001f);
    // keys: cell << 48 | caller's index << 16 | arrival slot
    int P = 1;
    while (P < n) P <<= 1;
    for (int k = threadIdx.x; k < P; k += kSortThreads) {
        unsigned long long kk = ~0ull;
        if (k < n) {
            const float y = v.ty[b0 + k], z = v.tz[b0 + k];
            const int iy = max(0, min((int)((y - ymin) * idy), ny - 1));
            const int iz = max(0, min((int)((z - zmin) * idz), nz - 1));
            const unsigned long long cell = (unsigned long long)(iz * ny + iy);
            kk = (cell << 48) | ((unsigned long long)(unsigned)v.tidx[b0 + k] << 16) | (unsigned long long)k;
        }
        key[k] = kk;
    }
    __syncthreads();
    // bitonic sort
    for (int size = 2; size <= P; size <<= 1) {
        for (int stride = size >> 1; stride > 0; stride >>= 1) {
            for (int t = threadIdx.x; t < (P >> 1); t += kSortThreads) {
                const int lo = 2 * t - (t & (stride - 1));
                const int hi = lo + stride;
                const bool up = ((lo & size) == 0);
                const unsigned long long a = key[lo], b = key[hi];
                if ((a > b) == up) { key[lo] = b; key[hi] = a; }
            }
            __syncthreads();
        }
    }
    // write sorted hits and the cell table
    const int ncell = ny * nz;
    for (int k = threadIdx.x; k < n; k += kSortThreads) {
        const unsigned long long kk = key[k];
        const int sl = (int)(kk & 0xffffull);
        v.sy[b0 + k] = v.ty[b0 + sl];
        v.sz[b0 + k] = v.tz[b0 + sl];
        v.sorig[b0 + k] = (int32_t)((kk >> 16) & 0xffffffffull);
        const int c = (int)(kk >> 48);
        const int cprev = k == 0 ? -1 : (int)(key[k - 1] >> 48);
        for (int q = cprev + 1; q <= c; q++) cs[q] = (uint16_t)k;
        if (k == n - 1)
            for (int q = c + 1; q <= ncell; q++) cs[q] = (uint16_t)n;
    }
    if (threadIdx.x == 0) {
        v.grid_f[bin] = make_float4(ymin, zmin, idy, idz);
        v.grid_n[bin] = make_int2(ny, nz);
    }
}

// ---------------------------------------------------------------------------------------------------------
// K2 neighbour finder.  One CTA per bin (task,row); a thread takes hits of the row.
// For hit h of row r: among up-candidates u (row r+D) and down-candidates d (row r-D) inside the windows,
// minimise D = (y0 - yhat)^2 + (z0 - zhat)^2 with (yhat, zhat) the point of the line d->u at x0;
// ties -> lowest caller's index of u, then of d.
// ---------------------------------------------------------------------------------------------------------
constexpr int kNfThreads = 128;

__global__ void __launch_bounds__(kNfThreads) k_neighbours(const View v, const __grid_constant__ Const c) {
    const int bin = blockIdx.x;
    const int nr = c.n_rows, D = c.p.link_step;
    const int r = bin % nr;
    const int b0 = v.bin_start[bin], n = v.bin_start[bin + 1] - b0;
    if (n == 0) return;
    if (r - D < 0 || r + D >= nr) {
        for (int k = threadIdx.x; k < n; k += kNfThreads) { v.link_up[b0 + k] = -1; v.link_dn[b0 + k] = -1; }
        return;
    }
    const float x0 = c.row_x[r], x1 = c.row_x[r + D], x2 = c.row_x[r - D];
    const float wyu = c.p.nf_slope_y * fabsf(x1 - x0) + c.p.nf_w0, wzu = c.p.nf_slope_z * fabsf(x1 - x0) + c.p.nf_w0;
    const float wyd = c.p.nf_slope_y * fabsf(x2 - x0) + c.p.nf_w0, wzd = c.p.nf_slope_z * fabsf(x2 - x0) + c.p.nf_w0;
    const float a = (x0 - x2) / (x1 - x2);
    const RowGrid gu = load_grid(v, bin + D), gd = load_grid(v, bin - D);
    const bool none = (v.bin_start[bin + D + 1] - gu.base == 0) || (v.bin_start[bin - D + 1] - gd.base == 0);
    for (int k = threadIdx.x; k < n; k += kNfThreads) {
        const int h = b0 + k;
        int bu = -1, bd = -1, bou = 0, bod = 0;
        float best = 0.f;
        if (!none) {
            const float y0 = v.sy[h], z0 = v.sz[h];
            GridIter iu;
            iu.start(gu, y0, z0, wyu, wzu);
            int u;
            while (iu.next(u)) {
                const float yu = v.sy[u], zu = v.sz[u];
                if (!(fabsf(yu - y0) <= wyu && fabsf(zu - z0) <= wzu)) continue;
                const int ou = v.sorig[u];
                GridIter id;
                id.start(gd, y0, z0, wyd, wzd);
                int d;
                while (id.next(d)) {
                    const float yd = v.sy[d], zd = v.sz[d];
                    if (!(fabsf(yd - y0) <= wyd && fabsf(zd - z0) <= wzd)) continue;
                    const float yh = yd + a * (yu - yd);
                    const float zh = zd + a * (zu - zd);
                    const float dy = y0 - yh, dz = z0 - zh;
                    const float dev = dy * dy + dz * dz;
                    bool take = bu < 0 || dev < best;
                    if (!take && dev == best) {
                        const int od = v.sorig[d];
                        take = ou < bou || (ou == bou && od < bod);
                    }
                    if (take) { best = dev; bu = u; bd = d; bou = ou; bod = v.sorig[d]; }
                }
            }
            if (!(bu >= 0 && best <= c.p.nf_dmax)) { bu = -1; bd = -1; }
        }
        v.link_up[h] = bu;
        v.link_dn[h] = bd;
    }
}

// ---------------------------------------------------------------------------------------------------------
// K3 cleaner + start-hit count.  clink_up[h] = link_up[h] if link_dn[link_up[h]] == h, else -1 (and the
// mirror image); one simultaneous pass.  A start hit has a cleaned up-link and no cleaned down-link.
// ---------------------------------------------------------------------------------------------------------
constexpr int kCleanThreads = 128;

__global__ void __launch_bounds__(kCleanThreads) k_clean(const View v) {
    __shared__ int nstart, nlink;
    const int bin = blockIdx.x;
    const int b0 = v.bin_start[bin], n = v.bin_start[bin + 1] - b0;
    if (threadIdx.x == 0) { nstart = 0; nlink = 0; }
    __syncthreads();
    int ns = 0, nl = 0;
    for (int k = threadIdx.x; k < n; k += kCleanThreads) {
        const int h = b0 + k;
        const int u = v.link_up[h], d = v.link_dn[h];
        const int cu = (u >= 0 && v.link_dn[u] == h) ? u : -1;
        const int cd = (d >= 0 && v.link_up[d] == h) ? d : -1;
        v.clink_up[h] = cu;
        v.clink_dn[h] = cd;
        ns += (cu >= 0 && cd < 0);
        nl += (cu >= 0);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { ns += __shfl_xor_sync(0xffffffffu, ns, o); nl += __shfl_xor_sync(0xffffffffu, nl, o); }
    if (lane_id() == 0 && (ns | nl)) { atomicAdd(&nstart, ns); atomicAdd(&nlink, nl); }
    __syncthreads();
    if (threadIdx.x == 0) {
        v.seed_count[bin] = nstart;
        if (nlink) atomicAdd(&v.cnt[CNT_LINKS], (unsigned long long)nlink);
    }
}

// ---------------------------------------------------------------------------------------------------------
// K4 start-hit compaction in canonical order (task, row, caller's index): warp ballot + prefix popcount
// collects the row's start hits, a rank by caller's index orders them.
// ---------------------------------------------------------------------------------------------------------
constexpr int kSeedThreads = 128;

__global__ void __launch_bounds__(kSeedThreads) k_seeds(const View v) {
    __shared__ int list_h[TPC_MAX_ROW_HITS];
    __shared__ int list_o[TPC_MAX_ROW_HITS];
    __shared__ int fill;
    const int bin = blockIdx.x;
    const int s0 = v.seed_start[bin], ns = v.seed_start[bin + 1] - s0;
    if (ns == 0) return;
    const int b0 = v.bin_start[bin], n = v.bin_start[bin + 1] - b0;
    if (threadIdx.x == 0) fill = 0;
    __syncthreads();
    for (int k0 = 0; k0 < n; k0 += kSeedThreads) {
        const int k = k0 + threadIdx.x;
        bool st = false;
        if (k < n) st = v.clink_up[b0 + k] >= 0 && v.clink_dn[b0 + k] < 0;
        const unsigned m = __ballot_sync(0xffffffffu, st);
        int basep = 0;
        if (lane_id() == 0 && m) basep = atomicAdd(&fill, __popc(m));
        basep = __shfl_sync(0xffffffffu, basep, 0);
        if (st) {
            const int p = basep + __popc(m & ((1u << lane_id()) - 1u));
            list_h[p] = b0 + k;
            list_o[p] = v.sorig[b0 + k];
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < ns; i += kSeedThreads) {
        const int o = list_o[i];
        int rank = 0;
        for (int j = 0; j < ns; j++) rank += (list_o[j] < o);
        if (s0 + rank < v.S_cap) { v.seeds[s0 + rank] = list_h[i]; v.seed_bin[s0 + rank] = bin; }
        else atomicOr((unsigned int*)&v.cnt[CNT_ERR], kErrSeedCapacity);
    }
}

}  // namespace tpc
