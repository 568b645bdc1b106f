// kf_kernels.cuh -- K5 tracklet constructor (float32 helix Kalman filter) and K6 tracklet selector.
// Every float expression is parenthesised exactly as DESIGN.md "O5" writes it and compiled with -fmad=false:
// the gates, windows and arg-mins then take the same decisions as the strict-float32 reference.
#pragma once
#include "common.cuh"

namespace tpc {

// Fit state: y, z, sin phi, tg lambda (dz/dS), q/pT and the lower triangle of the covariance.
struct Fit {
    float y, z, s, t, q;
    float c00, c10, c11, c20, c21, c22, c30, c31, c32, c33, c40, c41, c42, c43, c44;
    float chi2;
    int n;
};

__device__ __forceinline__ void fit_prior(Fit& f, const Const& c) {
    f.c00 = c.sigma_y2; f.c11 = c.sigma_z2; f.c22 = c.p.var_s; f.c33 = c.p.var_t; f.c44 = c.p.var_q;
    f.c10 = f.c20 = f.c21 = f.c30 = f.c31 = f.c32 = f.c40 = f.c41 = f.c42 = f.c43 = 0.f;
    f.chi2 = 0.f;
}

// Helix transport x -> x1.  false (fit untouched) if |sin phi| leaves [-s_max, s_max].
__device__ __forceinline__ bool fit_transport(Fit& f, float x, float x1, const Const& c) {
    const float kB = c.kB;
    const float dx = x1 - x;
    const float kap = kB * f.q;
    const float s = f.s, s1 = s + kap * dx;
    if (fabsf(s) > c.p.sin_max) return false;
    if (fabsf(s1) > c.p.sin_max) return false;
    const float c0 = sqrtf(1.f - s * s), c1 = sqrtf(1.f - s1 * s1);
    const float icc = 1.f / (c0 + c1), ic0 = 1.f / c0, ic1 = 1.f / c1;
    const float dy = dx * ((s + s1) * icc);
    const float dl2 = dx * dx + dy * dy;
    const float dl = (dx < 0.f) ? -sqrtf(dl2) : sqrtf(dl2);
    const float idl = 1.f / dl;
    const float u = kap * dl, u2 = u * u;
    const float c24 = 1.f / 24.f, c640 = 3.f / 640.f, c12 = 1.f / 12.f;
    const float dS = dl * (1.f + u2 * (c24 + u2 * c640));
    const float ccd = 1.f + (c0 * c1 + s * s1);
    // Jacobian rows y: (1 0 a 0 b), z: (0 1 cc d e), s: (0 0 1 0 ff)
    const float a = dx * ccd * icc * ic0 * ic1;
    const float b = kB * (dx * dx) * ccd * ic1 * icc * icc;
    const float cc = f.t * dy * ic0 * ic1;
    const float d = dS;
    const float e = f.t * ((dy * idl) * b + (kB * kap) * (dl * dl2) * c12);
    const float ff = kB * dx;
    f.y = f.y + dy; f.z = f.z + f.t * dS; f.s = s1;
    // M = F C, terms added in ascending column index of F
    const float m00 = f.c00 + a * f.c20 + b * f.c40;
    const float m02 = f.c20 + a * f.c22 + b * f.c42;
    const float m04 = f.c40 + a * f.c42 + b * f.c44;
    const float m10 = f.c10 + cc * f.c20 + d * f.c30 + e * f.c40;
    const float m11 = f.c11 + cc * f.c21 + d * f.c31 + e * f.c41;
    const float m12 = f.c21 + cc * f.c22 + d * f.c32 + e * f.c42;
    const float m13 = f.c31 + cc * f.c32 + d * f.c33 + e * f.c43;
    const float m14 = f.c41 + cc * f.c42 + d * f.c43 + e * f.c44;
    const float m20 = f.c20 + ff * f.c40, m21 = f.c21 + ff * f.c41, m22 = f.c22 + ff * f.c42;
    const float m23 = f.c32 + ff * f.c43, m24 = f.c42 + ff * f.c44;
    const float m30 = f.c30, m31 = f.c31, m32 = f.c32, m33 = f.c33, m34 = f.c43;
    const float m40 = f.c40, m41 = f.c41, m42 = f.c42, m43 = f.c43, m44 = f.c44;
    // C' = M F^T, lower triangle, terms added in ascending column index
    f.c00 = m00 + m02 * a + m04 * b;
    f.c10 = m10 + m12 * a + m14 * b;
    f.c11 = m11 + m12 * cc + m13 * d + m14 * e;
    f.c20 = m20 + m22 * a + m24 * b;
    f.c21 = m21 + m22 * cc + m23 * d + m24 * e;
    f.c22 = m22 + m24 * ff;
    f.c30 = m30 + m32 * a + m34 * b;
    f.c31 = m31 + m32 * cc + m33 * d + m34 * e;
    f.c32 = m32 + m34 * ff;
    f.c33 = m33;
    f.c40 = m40 + m42 * a + m44 * b;
    f.c41 = m41 + m42 * cc + m43 * d + m44 * e;
    f.c42 = m42 + m44 * ff;
    f.c43 = m43;
    f.c44 = m44;
    return true;
}

// gate value of a measurement against the predicted state
__device__ __forceinline__ float fit_gate(const Fit& f, float my, float mz, const Const& c) {
    const float ry = my - f.y, rz = mz - f.z;
    const float wy = 1.f / (f.c00 + c.sigma_y2);
    const float wz = 1.f / (f.c11 + c.sigma_z2);
    return (ry * ry) * wy + (rz * rz) * wz;
}

// two scalar updates, y then z
__device__ __forceinline__ void fit_update(Fit& f, float my, float mz, const Const& c) {
    {
        const float r = my - f.y;
        const float w = 1.f / (f.c00 + c.sigma_y2);
        const float k0 = f.c00, k1 = f.c10, k2 = f.c20, k3 = f.c30, k4 = f.c40;
        const float g0 = k0 * w, g1 = k1 * w, g2 = k2 * w, g3 = k3 * w, g4 = k4 * w;
        f.y = f.y + g0 * r; f.z = f.z + g1 * r; f.s = f.s + g2 * r; f.t = f.t + g3 * r; f.q = f.q + g4 * r;
        f.c00 = f.c00 - g0 * k0;
        f.c10 = f.c10 - g1 * k0; f.c11 = f.c11 - g1 * k1;
        f.c20 = f.c20 - g2 * k0; f.c21 = f.c21 - g2 * k1; f.c22 = f.c22 - g2 * k2;
        f.c30 = f.c30 - g3 * k0; f.c31 = f.c31 - g3 * k1; f.c32 = f.c32 - g3 * k2; f.c33 = f.c33 - g3 * k3;
        f.c40 = f.c40 - g4 * k0; f.c41 = f.c41 - g4 * k1; f.c42 = f.c42 - g4 * k2; f.c43 = f.c43 - g4 * k3;
        f.c44 = f.c44 - g4 * k4;
        f.chi2 = f.chi2 + (r * r) * w;
    }
    {
        const float r = mz - f.z;
        const float w = 1.f / (f.c11 + c.sigma_z2);
        const float k0 = f.c10, k1 = f.c11, k2 = f.c21, k3 = f.c31, k4 = f.c41;
        const float g0 = k0 * w, g1 = k1 * w, g2 = k2 * w, g3 = k3 * w, g4 = k4 * w;
        f.y = f.y + g0 * r; f.z = f.z + g1 * r; f.s = f.s + g2 * r; f.t = f.t + g3 * r; f.q = f.q + g4 * r;
        f.c00 = f.c00 - g0 * k0;
        f.c10 = f.c10 - g1 * k0; f.c11 = f.c11 - g1 * k1;
        f.c20 = f.c20 - g2 * k0; f.c21 = f.c21 - g2 * k1; f.c22 = f.c22 - g2 * k2;
        f.c30 = f.c30 - g3 * k0; f.c31 = f.c31 - g3 * k1; f.c32 = f.c32 - g3 * k2; f.c33 = f.c33 - g3 * k3;
        f.c40 = f.c40 - g4 * k0; f.c41 = f.c41 - g4 * k1; f.c42 = f.c42 - g4 * k2; f.c43 = f.c43 - g4 * k3;
        f.c44 = f.c44 - g4 * k4;
        f.chi2 = f.chi2 + (r * r) * w;
    }
    f.n++;
}

// best hit of bin (task,row) inside the window of the predicted state, or -1
__device__ __forceinline__ int fit_search(const Fit& f, const View& v, int bin, const Const& c) {
    if (v.bin_start[bin + 1] == v.bin_start[bin]) return -1;
    const float wy = fminf(fmaxf(c.p.win_nsigma * sqrtf(f.c00 + c.sigma_y2), c.p.win_min), c.p.win_max);
    const float wz = fminf(fmaxf(c.p.win_nsigma * sqrtf(f.c11 + c.sigma_z2), c.p.win_min), c.p.win_max);
    const RowGrid g = load_grid(v, bin);
    GridIter it;
    it.start(g, f.y, f.z, wy, wz);
    int best = -1, bo = 0, h;
    float gb = 0.f;
    while (it.next(h)) {
        const float y = v.sy[h], z = v.sz[h];
        if (!(fabsf(y - f.y) <= wy && fabsf(z - f.z) <= wz)) continue;
        const float gv = fit_gate(f, y, z, c);
        bool take = best < 0 || gv < gb;
        int o = 0;
        if (!take && gv == gb) { o = v.sorig[h]; take = o < bo; }
        else if (take) o = v.sorig[h];
        if (take) { gb = gv; best = h; bo = o; }
    }
    if (best < 0) return -1;
    return (gb <= c.p.chi2_ext) ? best : -1;
}

__device__ __forceinline__ int32_t* table_ptr(const View& v, int i, int nr) {
    return v.tl_table + (size_t)(i / kChunk) * nr * kChunk + (i % kChunk);
}

// ---------------------------------------------------------------------------------------------------------
// K5: one thread per start hit (grid-stride).  Up pass along the cleaned links, then extension by search;
// down pass = fresh fit from the top hit through everything recorded, searching the empty rows.
// ---------------------------------------------------------------------------------------------------------
constexpr int kKfThreads = 128;

__global__ void __launch_bounds__(kKfThreads) k_construct(const View v, const __grid_constant__ Const c) {
    const int S = min(v.seed_start[v.n_bins], v.S_cap);
    const int nr = c.n_rows;
    unsigned long long visits = 0;
    for (int i = blockIdx.x * kKfThreads + threadIdx.x; i < S; i += gridDim.x * kKfThreads) {
        int32_t* tab = table_ptr(v, i, nr);  // tab[row * kChunk]
        const int h0 = v.seeds[i];
        const int bin0 = v.seed_bin[i];
        const int r0 = bin0 % nr;
        const int tb = bin0 - r0;  // first bin of this task
        const int h1 = v.clink_up[h0];
        Fit f;
        {
            const int D = c.p.link_step;
            const float dx = c.row_x[r0 + D] - c.row_x[r0];
            const float y0 = v.sy[h0], z0 = v.sz[h0];
            const float dy = v.sy[h1] - y0, dz = v.sz[h1] - z0;
            const float dl = sqrtf(dx * dx + dy * dy);
            f.y = y0; f.z = z0; f.s = dy / dl; f.t = dz / dl; f.q = 0.f;
            fit_prior(f, c); f.n = 1;
        }
        tab[r0 * kChunk] = h0;
        float ss = f.s, st = f.t, sq = f.q;  // direction / curvature at the last accepted update
        int top = r0;
        // ---- up pass ----
        {
            bool follow = true;
            int cur = h1, rcur = r0 + c.p.link_step, miss = 0;
            float xc = c.row_x[r0];
            for (int row = r0 + 1; row < nr; row++) {
                if (!fit_transport(f, xc, c.row_x[row], c)) break;
                visits++;
                xc = c.row_x[row];
                int acc = -1;
                bool stop = false;
                if (follow && row < rcur) {
                    // in-between row of a step-2 link: nothing to do
                } else {
                    if (follow) {
                        const float my = v.sy[cur], mz = v.sz[cur];
                        if (fit_gate(f, my, mz, c) <= c.p.chi2_link) {
                            acc = cur;
                            cur = v.clink_up[cur];
                            rcur += c.p.link_step;
                            if (cur < 0) follow = false;
                        } else {
                            follow = false;
                        }
                    }
                    if (acc < 0) {  // extend by search (also the row where following just failed)
                        if (fabsf(f.y) > c.row_x[row] * c.tan_half_angle + c.p.edge_margin) stop = true;
                        else {
                            acc = fit_search(f, v, tb + row, c);
                            if (acc >= 0) miss = 0;
                            else if (++miss > c.p.max_gap) stop = true;
                        }
                    }
                }
                if (stop) break;
                tab[row * kChunk] = acc;
                if (acc >= 0) {
                    fit_update(f, v.sy[acc], v.sz[acc], c);
                    ss = f.s; st = f.t; sq = f.q; top = row;
                }
            }
        }
        // ---- down pass ----
        int first = top, nh = 1;
        float py, pz, ps, pt, pq, pchi2;
        {
            const int ht = tab[top * kChunk];
            f.y = v.sy[ht]; f.z = v.sz[ht]; f.s = ss; f.t = st; f.q = sq;
            fit_prior(f, c); f.n = 1;
            py = f.y; pz = f.z; ps = f.s; pt = f.t; pq = f.q; pchi2 = f.chi2;
            int miss = 0;
            float xc = c.row_x[top];
            int row = top - 1;
            for (; row >= 0; row--) {
                if (!fit_transport(f, xc, c.row_x[row], c)) break;
                visits++;
                xc = c.row_x[row];
                const bool below = row < r0;
                int acc = -1;
                bool searched = false;
                if (!below) {
                    const int hr = tab[row * kChunk];
                    if (hr >= 0) {
                        if (fit_gate(f, v.sy[hr], v.sz[hr], c) <= c.p.chi2_link) acc = hr;
                    } else searched = true;
                } else searched = true;
                if (searched) {
                    if (below && fabsf(f.y) > c.row_x[row] * c.tan_half_angle + c.p.edge_margin) break;
                    acc = fit_search(f, v, tb + row, c);
                    if (acc >= 0) miss = 0;
                    else if (below && ++miss > c.p.max_gap) break;
                }
                tab[row * kChunk] = acc;
                if (acc >= 0) {
                    fit_update(f, v.sy[acc], v.sz[acc], c);
                    py = f.y; pz = f.z; ps = f.s; pt = f.t; pq = f.q; pchi2 = f.chi2;
                    first = row; nh = f.n;
                }
            }
            // rows the pass never reached keep nothing (only rows >= r0 can hold stale up-pass entries)
            for (; row >= r0; row--) tab[row * kChunk] = -1;
        }
        v.tl_rows[i] = first | (top << 8) | (nh << 16);
        const int sc = v.S_cap;
        v.tl_par[i] = py; v.tl_par[sc + i] = pz; v.tl_par[2 * sc + i] = ps; v.tl_par[3 * sc + i] = pt;
        v.tl_par[4 * sc + i] = pq; v.tl_par[5 * sc + i] = pchi2;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) visits += __shfl_xor_sync(0xffffffffu, visits, o);
    if (lane_id() == 0 && visits) atomicAdd(&v.cnt[CNT_ROW_VISITS], visits);
}

// ---------------------------------------------------------------------------------------------------------
// K6 selector.  key = n_hits << 24 | (2^24 - 1 - id within the task): larger = more hits, then lower
// canonical id.  owner[hit] = max key over tracklets (n_hits >= min_tracklet_hits) holding the hit.
// One warp per table chunk: lane = tracklet, loop over rows -> coalesced table reads.
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t tl_key(const View& v, int i, int nh, int nr) {
    const int bin = v.seed_bin[i];
    const int id_in_task = i - v.seed_start[bin - bin % nr];
    return ((uint32_t)nh << 24) | (uint32_t)(0xffffff - id_in_task);
}

constexpr int kSelThreads = 128;

__global__ void __launch_bounds__(kSelThreads) k_claim(const View v, const __grid_constant__ Const c) {
    const int S = min(v.seed_start[v.n_bins], v.S_cap);
    const int nr = c.n_rows;
    const int chunk = (blockIdx.x * kSelThreads + threadIdx.x) / 32;
    const int i = chunk * kChunk + lane_id();
    if (chunk * kChunk >= S) return;
    int first = nr, last = -1, nh = 0;
    uint32_t key = 0;
    if (i < S) {
        const int pk = v.tl_rows[i];
        nh = pk >> 16;
        if (nh >= c.p.min_tracklet_hits) { first = pk & 0xff; last = (pk >> 8) & 0xff; key = tl_key(v, i, nh, nr); }
    }
    int lo = first, hi = last;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { lo = min(lo, __shfl_xor_sync(0xffffffffu, lo, o)); hi = max(hi, __shfl_xor_sync(0xffffffffu, hi, o)); }
    const int32_t* tab = v.tl_table + (size_t)chunk * nr * kChunk + lane_id();
    int cnt = 0;
    for (int row = lo; row <= hi; row++) {
        if (row < first || row > last) continue;
        const int h = tab[row * kChunk];
        if (h >= 0) { atomicMax(&v.owner[h], key); cnt++; }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
    if (lane_id() == 0 && cnt) atomicAdd(&v.cnt[CNT_TL_HITS], (unsigned long long)cnt);
}

__global__ void __launch_bounds__(kSelThreads) k_count_owned(const View v, const __grid_constant__ Const c) {
    const int S = min(v.seed_start[v.n_bins], v.S_cap);
    const int nr = c.n_rows;
    const int chunk = (blockIdx.x * kSelThreads + threadIdx.x) / 32;
    const int i = chunk * kChunk + lane_id();
    if (chunk * kChunk >= S) return;
    int first = nr, last = -1, nh = 0;
    uint32_t key = 0;
    if (i < S) {
        const int pk = v.tl_rows[i];
        nh = pk >> 16;
        if (nh >= c.p.min_tracklet_hits) { first = pk & 0xff; last = (pk >> 8) & 0xff; key = tl_key(v, i, nh, nr); }
    }
    int lo = first, hi = last;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { lo = min(lo, __shfl_xor_sync(0xffffffffu, lo, o)); hi = max(hi, __shfl_xor_sync(0xffffffffu, hi, o)); }
    const int32_t* tab = v.tl_table + (size_t)chunk * nr * kChunk + lane_id();
    int own = 0;
    for (int row = lo; row <= hi; row++) {
        if (row < first || row > last) continue;
        const int h = tab[row * kChunk];
        if (h >= 0 && v.owner[h] == key) own++;
    }
    if (i < S) {
        const int keep = own >= c.p.min_track_hits;
        v.tl_keep[i] = keep;
        v.tl_nown[i] = keep ? own : 0;
    }
}

// track / hit offsets of every event (tracks of one event are contiguous: seeds are ordered by task)
__global__ void k_event_offsets(const View v, int bins_per_event) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e > v.n_events) return;
    const int S = min(v.seed_start[v.n_bins], v.S_cap);
    const int s = min(v.seed_start[e * bins_per_event], S);
    v.ev_off[e] = v.trk_scan[s];
    v.ev_off[v.n_events + 1 + e] = v.hit_scan[s];
    if (e == v.n_events) { v.cnt[CNT_TRACKS] = (unsigned long long)v.trk_scan[s]; v.cnt[CNT_TRACK_HITS] = (unsigned long long)v.hit_scan[s]; }
}

__global__ void __launch_bounds__(kSelThreads) k_write_tracks(const View v, const __grid_constant__ Const c) {
    const int S = min(v.seed_start[v.n_bins], v.S_cap);
    const int nr = c.n_rows;
    const int chunk = (blockIdx.x * kSelThreads + threadIdx.x) / 32;
    const int i = chunk * kChunk + lane_id();
    if (chunk * kChunk >= S) return;
    int first = nr, last = -1, nh = 0, ho = 0;
    uint32_t key = 0;
    if (i < S && v.tl_keep[i]) {
        const int pk = v.tl_rows[i];
        nh = pk >> 16; first = pk & 0xff; last = (pk >> 8) & 0xff; key = tl_key(v, i, nh, nr);
        const int ti = v.trk_scan[i];
        ho = v.hit_scan[i];
        const int bin = v.seed_bin[i];
        const int task = bin / nr;
        const int e = task / c.n_sectors;
        const int sc = v.S_cap;
        v.o_sector[ti] = task % c.n_sectors;
        v.o_first_hit[ti] = ho - v.ev_off[v.n_events + 1 + e];
        v.o_n_hits[ti] = v.tl_nown[i];
        v.o_ndf[ti] = 2 * nh - 5;
        v.o_x[ti] = c.row_x[first];
        v.o_y[ti] = v.tl_par[i]; v.o_z[ti] = v.tl_par[sc + i]; v.o_sinphi[ti] = v.tl_par[2 * sc + i];
        v.o_tgl[ti] = v.tl_par[3 * sc + i]; v.o_qpt[ti] = v.tl_par[4 * sc + i]; v.o_chi2[ti] = v.tl_par[5 * sc + i];
    }
    int lo = first, hi = last;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { lo = min(lo, __shfl_xor_sync(0xffffffffu, lo, o)); hi = max(hi, __shfl_xor_sync(0xffffffffu, hi, o)); }
    const int32_t* tab = v.tl_table + (size_t)chunk * nr * kChunk + lane_id();
    for (int row = lo; row <= hi; row++) {
        if (row < first || row > last) continue;
        const int h = tab[row * kChunk];
        if (h >= 0 && v.owner[h] == key) v.o_hit_idx[ho++] = v.sorig[h];
    }
}

}  // namespace tpc
