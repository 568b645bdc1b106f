// merge_kernels.cuh -- O9: links between the track segments of one particle across sector borders
// ("global reconstruction ... merged together").
//
// Segment A (outer state of its refit at pad row r_A) may continue in segment B of a neighbouring sector of the
// same side whose first fitted row r_B obeys 1 <= r_B - r_A <= 1 + max_gap.  A's outer state is turned into B's
// frame, moved along its helix to x = row_x[r_B] (state only, the transport formulas of DESIGN.md "O5") and
// compared with B's parameters there.  next(A) = arg min_B D, prev(B) = arg min_A D, ties -> lowest track index;
// a link is kept when mutual.  The refitted tracks are listed by (sector task, first fitted row) -- counted by K7,
// scanned, scattered -- so that a segment meets only the few candidates in the 1 + max_gap rows above its outer row.
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

constexpr unsigned long long kNoLink = ~0ull;

// tracks with a refit -> lists by (task, first fitted row); dn_count was filled by k_refit, dn_start is its scan
__global__ void __launch_bounds__(128) k_merge_scatter(const View v, int nr, int32_t* list, unsigned long long* pvkey) {
    const int T = (int)v.cnt[CNT_TRACKS];
    const int a = blockIdx.x * 128 + threadIdx.x;
    if (a >= T) return;
    pvkey[a] = kNoLink;
    const int rows = v.trk_rows[a];
    if (rows < 0) return;
    const int bin = v.trk_task[a] * nr + (rows & 0xff);
    list[v.dn_start[bin] + atomicAdd(&v.dn_fill[bin], 1)] = a;
}

// One thread per segment a: the candidates b are the segments of the two neighbouring sectors whose first fitted
// row lies 1 .. 1 + max_gap rows above a's outer row (taken from the (task, row) lists).  Every candidate pair is
// scored once: it competes for next(a) in a register and for prev(b) with an atomicMin.  Keys are
// (bits of D) << 32 | track index: D >= +0, so the order of the keys is the order of (D, index) -- the lowest index
// wins a tie, as the reference's ascending loops do.
__global__ void __launch_bounds__(128) k_merge_pairs(const View v, const __grid_constant__ Const c, const int32_t* list,
                                                     unsigned long long* nxkey, unsigned long long* pvkey) {
    const int T = (int)v.cnt[CNT_TRACKS];
    const int a = blockIdx.x * 128 + threadIdx.x;
    if (a >= T) return;
    unsigned long long best = kNoLink;
    const int rows_a = v.trk_rows[a];
    const int ns = c.n_sectors, nr = c.n_rows, half = ns >> 1;
    if (rows_a >= 0 && ns >= 4 && !(ns & 1)) {
        const int task = v.trk_task[a];
        const int ev = task / ns, s = task - ev * ns, side = s / half, k = s - side * half;
        const int k_lo = (k + half - 1) % half, k_hi = (k + 1) % half;   // the sectors before / after a's
        const int r_out = (rows_a >> 8) & 0xff;
        const int r0 = r_out + 1, r1 = min(r_out + 1 + c.p.merge_max_gap, nr - 1);
        for (int j = 0; j < 2; j++) {
            if (j == 1 && k_hi == k_lo) break;   // two sectors per side: one neighbour
            const int kb = j == 0 ? k_hi : k_lo;
            const int other = ev * ns + side * half + kb;
            if (r0 > r1) break;
            const int p0 = v.dn_start[other * nr + r0], p1 = v.dn_start[other * nr + r1 + 1];
            for (int p = p0; p < p1; p++) {
                const int b = list[p];
                float D;
                if (!merge_score(v, c, a, b, rows_a, v.trk_rows[b], kb == k_hi, D)) continue;
                const unsigned long long d = (unsigned long long)__float_as_uint(D) << 32;
                best = min(best, d | (unsigned)b);
                atomicMin(&pvkey[b], d | (unsigned)a);
            }
        }
    }
    nxkey[a] = best;
}

// keep the mutual links; indices become event-local
__global__ void __launch_bounds__(128) k_merge_mutual(const View v, const __grid_constant__ Const c, const unsigned long long* nxkey,
                                                      const unsigned long long* pvkey) {
    const int T = (int)v.cnt[CNT_TRACKS];
    const int a = blockIdx.x * 128 + threadIdx.x;
    if (a >= T) return;
    const int e0 = v.ev_off[v.trk_task[a] / c.n_sectors];
    const unsigned long long kn = nxkey[a], kp = pvkey[a];
    const int b = kn == kNoLink ? -1 : (int)(kn & 0xffffffffu), p = kp == kNoLink ? -1 : (int)(kp & 0xffffffffu);
    const bool fwd = b >= 0 && pvkey[b] != kNoLink && (int)(pvkey[b] & 0xffffffffu) == a;
    const bool bwd = p >= 0 && nxkey[p] != kNoLink && (int)(nxkey[p] & 0xffffffffu) == a;
    v.o_next[a] = fwd ? b - e0 : -1;
    v.o_prev[a] = bwd ? p - e0 : -1;
}

// global track = chain of linked segments, named by its first segment.  A link leads to a higher pad row, so a
// chain is at most n_rows long and never closes on itself; n_sectors / 2 links at most in practice.
__global__ void __launch_bounds__(128) k_merge_chain(const View v, int n_sectors) {
    const int T = (int)v.cnt[CNT_TRACKS];
    const int a = blockIdx.x * 128 + threadIdx.x;
    if (a >= T) return;
    const int e0 = v.ev_off[v.trk_task[a] / n_sectors];   // o_prev holds event-local indices
    int h = a - e0;
    for (int p = v.o_prev[e0 + h]; p >= 0; p = v.o_prev[e0 + h]) h = p;
    v.o_global[a] = h;
}

}  // namespace tpc
