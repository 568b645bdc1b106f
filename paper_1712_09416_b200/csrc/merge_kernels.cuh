// merge_kernels.cuh -- O9: links between the track segments of one particle across sector borders
// ("global reconstruction ... merged together").
//
// Segment A (outer state of its refit at pad row r_A) may continue in segment B of a neighbouring sector of the
// same side whose first fitted row r_B obeys 1 <= r_B - r_A <= 1 + max_gap.  A's outer state is turned into B's
// frame, moved along its helix to x = row_x[r_B] (state only, the transport formulas of DESIGN.md "O5") and
// compared with B's parameters there.  next(A) = arg min_B D, prev(B) = arg min_A D, ties -> lowest track index;
// a link is kept when mutual.  One thread per track; the tracks of a sector task are contiguous (canonical order),
// so the threads of a warp walk the same candidate ranges and their loads are broadcasts.
#pragma once
#include "common.cuh"

namespace tpc {

// score of the ordered pair (a -> b); false when the pair is not a candidate.  Written as the reference
// parenthesises it (-fmad=false): the box tests and the arg min then decide identically.
__device__ __forceinline__ bool merge_score(const View& v, const Const& c, int a, int b, int rows_a, int rows_b, bool b_is_next,
                                            float& D) {
    const int gap = (rows_b & 0xff) - ((rows_a >> 8) & 0xff);
    if (gap < 1 || gap > 1 + c.p.merge_max_gap) return false;
    const float xa = v.o_xo[a], ya = v.o_yo[a], za = v.o_zo[a], s0 = v.o_so[a], t0 = v.o_to[a], q0 = v.o_qo[a];
    const float smax = c.p.sin_max;
    const float cd = c.merge_cd;
    const float sn = b_is_next ? 0.f - c.merge_sd : c.merge_sd;   // turn by alpha_A - alpha_B
    if (fabsf(s0) > smax) return false;
    const float c0a = sqrtf(1.f - s0 * s0);
    const float x1 = xa * cd - ya * sn;
    const float y1 = xa * sn + ya * cd;
    const float s1 = s0 * cd + c0a * sn;
    const float xb = v.o_x[b];
    const float dx = xb - x1;
    const float kap = c.kB * q0;
    const float s2 = s1 + kap * dx;
    if (fabsf(s1) > smax || fabsf(s2) > smax) return false;
    const float c1 = sqrtf(1.f - s1 * s1), c2 = sqrtf(1.f - s2 * s2);
    const float dy = dx * ((s1 + s2) * (1.f / (c1 + c2)));
    const float dl2 = dx * dx + dy * dy;
    const float adl = sqrtf(dl2);
    const float dl = (dx < 0.f) ? 0.f - adl : adl;
    const float u = kap * dl, u2 = u * u;
    const float dS = dl * (1.f + u2 * (1.f / 24.f + u2 * (3.f / 640.f)));
    const float y2 = y1 + dy, z2 = za + t0 * dS;
    const float ey = y2 - v.o_y[b], ez = z2 - v.o_z[b], es = s2 - v.o_sinphi[b], et = t0 - v.o_tgl[b];
    const float ty = c.p.merge_dy, tz = c.p.merge_dz, ts = c.p.merge_ds, tt = c.p.merge_dt;
    if (!(fabsf(ey) <= ty && fabsf(ez) <= tz && fabsf(es) <= ts && fabsf(et) <= tt)) return false;
    const float ny = ey * (1.f / ty), nz = ez * (1.f / tz), ns = es * (1.f / ts), nt = et * (1.f / tt);
    D = ((ny * ny + nz * nz) + ns * ns) + nt * nt;
    return true;
}

// first track of sector task `task` (tracks are ordered by task)
__device__ __forceinline__ int task_track0(const View& v, int task, int nr, int S) {
    return v.trk_scan[min(v.seed_start[task * nr], S)];
}

// NEXT: thread a looks for its best continuation b;  !NEXT: thread b looks for its best predecessor a
template <bool NEXT>
__global__ void __launch_bounds__(128) k_merge_best(const View v, const __grid_constant__ Const c, int32_t* best) {
    const int T = (int)v.cnt[CNT_TRACKS];
    const int me = blockIdx.x * 128 + threadIdx.x;
    if (me >= T) return;
    int res = -1;
    const int rows_me = v.trk_rows[me];
    const int ns = c.n_sectors, nr = c.n_rows, half = ns >> 1;
    if (rows_me >= 0 && ns >= 4 && !(ns & 1)) {
        const int S = min(v.seed_start[v.n_bins], v.S_cap);
        const int task = v.trk_task[me];
        const int ev = task / ns, s = task - ev * ns, side = s / half, k = s - side * half;
        const int k_lo = (k + half - 1) % half, k_hi = (k + 1) % half;   // the sectors before / after mine
        // candidate ranges in ascending track order (a strict < then keeps the lowest index on ties)
        int kk[2] = {min(k_lo, k_hi), max(k_lo, k_hi)};
        float bd = 0.f;
        for (int j = 0; j < 2; j++) {
            if (j == 1 && kk[1] == kk[0]) break;   // half == 2: one neighbour only
            const int other = ev * ns + side * half + kk[j];
            // the other sector is "next" of mine when it follows mine in azimuth
            const bool other_is_next = kk[j] == k_hi, other_is_prev = kk[j] == k_lo;
            const int t0 = task_track0(v, other, nr, S), t1 = task_track0(v, other + 1, nr, S);
            for (int o = t0; o < t1; o++) {
                const int rows_o = v.trk_rows[o];
                if (rows_o < 0) continue;
                float D;
                const bool ok = NEXT ? merge_score(v, c, me, o, rows_me, rows_o, other_is_next, D)
                                     : merge_score(v, c, o, me, rows_o, rows_me, other_is_prev, D);
                if (ok && (res < 0 || D < bd)) { res = o; bd = D; }
            }
        }
    }
    best[me] = res;
}

// keep the mutual links; indices become event-local
__global__ void __launch_bounds__(128) k_merge_mutual(const View v, const __grid_constant__ Const c, const int32_t* nx, const int32_t* pv) {
    const int T = (int)v.cnt[CNT_TRACKS];
    const int a = blockIdx.x * 128 + threadIdx.x;
    if (a >= T) return;
    const int e = v.trk_task[a] / c.n_sectors;
    const int e0 = v.ev_off[e];
    const int b = nx[a], p = pv[a];
    v.o_next[a] = (b >= 0 && pv[b] == a) ? b - e0 : -1;
    v.o_prev[a] = (p >= 0 && nx[p] == a) ? p - e0 : -1;
}

}  // namespace tpc
