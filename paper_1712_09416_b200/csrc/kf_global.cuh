// kf_global.cuh -- O10: one fit per global track = chain of track segments linked across sector borders (DESIGN.md
// "O10", SURVEY.md 8(f).2 "... then refit"; "merged together for global reconstruction").
//
// One lane per chain (its first segment), as a state machine that advances ONE pad row -- or one sector border -- per
// loop trip, like k_refit.  Up pass as O8 through the first segment; at the top hit of a segment the fit (state and
// covariance) is turned into the next segment's frame (fit_rotate), moved in one transport step to the row of that
// segment's first hit, updated with it, and goes on row by row.  Down pass: fresh fit at the last hit the up pass
// used, the same way back.  A lone segment's global fit is its O8 refit (the arithmetic would be the same); a segment
// that is not the first of its chain carries none.
#pragma once
#include "common.cuh"
#include "kf_kernels.cuh"

namespace tpc {

// the fit, given at x in one sector's frame, in the frame of a neighbouring sector whose axis is turned by the angle
// of sine sn, cosine cd; x becomes the point's abscissa there.  false: fit untouched.
__device__ __forceinline__ bool fit_rotate(Fit& f, float& x, float sn, float cd, const Const& c) {
    const float s = f.s;
    if (fabsf(s) > c.p.sin_max) return false;
    const float cc = sqrtf(1.f - s * s);
    const float s1 = s * cd + cc * sn;
    if (fabsf(s1) > c.p.sin_max) return false;
    const float c1 = sqrtf(1.f - s1 * s1);
    const float ic1 = 1.f / c1;
    const float kap = c.kB * f.q;
    const float jyy = cd + sn * (s1 * ic1);
    const float jzy = (f.t * sn) * ic1;
    const float jsy = kap * sn;
    const float jss = cd - (s * (1.f / cc)) * sn;
    const float x1 = x * cd - f.y * sn, y1 = x * sn + f.y * cd;
    x = x1; f.y = y1; f.s = s1;
    // M = J C (terms in ascending column of J), C' = M J^T (lower triangle, terms in ascending column)
    const float m00 = jyy * f.c00;
    const float m10 = jzy * f.c00 + f.c10, m11 = jzy * f.c10 + f.c11;
    const float m20 = jsy * f.c00 + jss * f.c20, m21 = jsy * f.c10 + jss * f.c21, m22 = jsy * f.c20 + jss * f.c22;
    const float m30 = f.c30, m32 = f.c32, m40 = f.c40, m42 = f.c42;
    f.c00 = m00 * jyy;
    f.c10 = m10 * jyy; f.c11 = m10 * jzy + m11;
    f.c20 = m20 * jyy; f.c21 = m20 * jzy + m21; f.c22 = m20 * jsy + m22 * jss;
    f.c30 = m30 * jyy; f.c31 = m30 * jzy + f.c31; f.c32 = m30 * jsy + m32 * jss;
    f.c40 = m40 * jyy; f.c41 = m40 * jzy + f.c41; f.c42 = m40 * jsy + m42 * jss;
    return true;
}

constexpr int kGfThreads = 128;

// lone segments and segments that are not the first of their chain get their entries here; the first segments of
// chains are listed (any order) for k_global_fit
__global__ void __launch_bounds__(kGfThreads) k_global_prep(const View v, int32_t* list) {
    const int T = (int)v.cnt[CNT_TRACKS];
    const int a = blockIdx.x * kGfThreads + threadIdx.x;
    if (a >= T) return;
    const bool head = v.o_prev[a] < 0, fitted = v.trk_rows[a] >= 0;
    if (head && fitted && v.o_next[a] >= 0) { list[(int)atomicAdd(&v.kf_cursor[1], 1ull)] = a; return; }
    const bool lone = head && fitted;   // its global fit is its refit
    v.o_gx[a] = lone ? v.o_x[a] : 0.f; v.o_gy[a] = lone ? v.o_y[a] : 0.f; v.o_gz[a] = lone ? v.o_z[a] : 0.f;
    v.o_gs[a] = lone ? v.o_sinphi[a] : 0.f; v.o_gt[a] = lone ? v.o_tgl[a] : 0.f; v.o_gq[a] = lone ? v.o_qpt[a] : 0.f;
    v.o_gchi2[a] = lone ? v.o_chi2[a] : 0.f;
    v.o_gndf[a] = lone ? v.o_ndf[a] : 0; v.o_gnhits[a] = lone ? (v.o_ndf[a] + 5) / 2 : 0;
    v.o_gsector[a] = lone ? v.o_sector[a] : -1;
}

// persistent: a lane takes a chain from the list, runs its up and down pass one row (or one border) per trip, and takes
// the next one
__global__ void __launch_bounds__(kGfThreads) k_global_fit(const View v, const __grid_constant__ Const c, const int32_t* list) {
    const int n_chains = (int)v.kf_cursor[1];
    const int lane = lane_id();
    const int ns = c.n_sectors, half = ns >> 1;
    // turn from segment p's sector to segment b's: -sin for the next sector in azimuth
    auto turn = [&](int p, int b) {
        const int dk = ((v.o_sector[b] % half) - (v.o_sector[p] % half) + half) % half;
        return dk == 1 ? 0.f - c.merge_sd : c.merge_sd;
    };
    Fit f;
    f.n = 0; f.chi2 = 0.f;
    float xc = 0.f;
    float s_s = 0.f, s_t = 0.f, s_q = 0.f, ty = 0.f, tz = 0.f;   // up pass right after its last update; the hit of that update
    int b_top = 0, j_top = 0, r_top = 0;
    float p0 = 0.f, p1 = 0.f, p2 = 0.f, p3 = 0.f, p4 = 0.f, p5 = 0.f;
    int rref = 0, nfit = 0, b_end = 0;
    int a = 0, e0 = 0, ph = 0, b = 0, h0 = 0, m = 0, j = 0, row = 0, nrow = -1;
    float ny = 0.f, nz = 0.f;                                   // the hit at position j of segment b (read ahead)
    auto load_hit = [&]() {
        nrow = -1;
        if (j >= 0 && j < m) { const float2 hn = v.o_hit_yz[h0 + j]; ny = hn.x; nz = hn.y; nrow = v.o_hit_row[h0 + j]; }
    };
    auto enter = [&](int seg) { b = seg; h0 = v.trk_hit0[seg]; m = v.o_n_hits[seg]; };
    bool more = true;
    for (;;) {
        const unsigned idle = __ballot_sync(kFull, ph == 0);
        if (idle && more) {
            int k0 = 0;
            if (lane == 0) k0 = (int)atomicAdd(&v.kf_cursor[3], (unsigned long long)__popc(idle));
            k0 = __shfl_sync(kFull, k0, 0);
            if (k0 >= n_chains) more = false;
            const int k = k0 + __popc(idle & lanemask_lt());
            if (ph == 0 && k < n_chains) {
                a = list[k];
                e0 = v.ev_off[v.trk_task[a] / ns];
                enter(a);
                const float2 a0 = v.o_hit_yz[h0], a1 = v.o_hit_yz[h0 + 1];
                const int r0 = v.o_hit_row[h0], r1 = v.o_hit_row[h0 + 1];
                const float dx = c.row_x[r1] - c.row_x[r0];
                const float dy = a1.x - a0.x, dz = a1.y - a0.y;
                const float dl = sqrtf(dx * dx + dy * dy);
                f.y = a0.x; f.z = a0.y; f.s = dy / dl; f.t = dz / dl; f.q = 0.f;
                fit_prior(f, c); f.n = 1;
                s_s = f.s; s_t = f.t; s_q = f.q; ty = a0.x; tz = a0.y; b_top = a; j_top = 0; r_top = r0;
                row = r0; xc = c.row_x[r0]; j = 1; load_hit();
                ph = 1;
            }
        }
        if (__all_sync(kFull, ph == 0)) break;
        bool upd = false, end = false;
        if (ph == 1) {
            if (j < m) {   // inside the segment: one pad row
                row++;
                end = !fit_transport(f, xc, c.row_x[row], c);
                if (!end) { xc = c.row_x[row]; upd = row == nrow; }
            } else {       // at the segment's top hit: across the border into the next segment, if there is one
                const int nb = v.o_next[b] < 0 ? -1 : e0 + v.o_next[b];
                end = nb < 0;
                if (!end) end = !fit_rotate(f, xc, turn(b, nb), c.merge_cd, c);
                if (!end) {
                    enter(nb); j = 0; load_hit();
                    const float xb = c.row_x[nrow];
                    if (xb != xc) end = !fit_transport(f, xc, xb, c);
                    if (!end) { xc = xb; row = nrow; upd = true; }
                }
            }
        } else if (ph == 2) {
            if (j >= 0) {
                row--;
                end = !fit_transport(f, xc, c.row_x[row], c);
                if (!end) { xc = c.row_x[row]; upd = row == nrow; }
            } else {
                const int pb = (b == a || v.o_prev[b] < 0) ? -1 : e0 + v.o_prev[b];
                end = pb < 0;
                if (!end) end = !fit_rotate(f, xc, 0.f - turn(pb, b), c.merge_cd, c);
                if (!end) {
                    enter(pb); j = m - 1; load_hit();
                    const float xb = c.row_x[nrow];
                    if (xb != xc) end = !fit_transport(f, xc, xb, c);
                    if (!end) { xc = xb; row = nrow; upd = true; }
                }
            }
        }
        __syncwarp();
        if (upd) {
            const float iwy = 1.f / (f.c00 + c.sigma_y2);
            fit_update(f, ny, nz, iwy, c);
            if (ph == 1) { s_s = f.s; s_t = f.t; s_q = f.q; ty = ny; tz = nz; b_top = b; j_top = j; r_top = row; j++; }
            else { p0 = f.y; p1 = f.z; p2 = f.s; p3 = f.t; p4 = f.q; p5 = f.chi2; rref = row; nfit = f.n; b_end = b; j--; }
            load_hit();
        }
        __syncwarp();
        if (end) {
            if (ph == 1) {   // fresh fit at the last hit the up pass used
                f.y = ty; f.z = tz; f.s = s_s; f.t = s_t; f.q = s_q;
                fit_prior(f, c); f.n = 1;
                p0 = ty; p1 = tz; p2 = s_s; p3 = s_t; p4 = s_q; p5 = 0.f; rref = r_top; nfit = 1; b_end = b_top;
                enter(b_top); row = r_top; xc = c.row_x[r_top]; j = j_top - 1; load_hit();
                ph = 2;
            } else {
                v.o_gx[a] = c.row_x[rref]; v.o_gy[a] = p0; v.o_gz[a] = p1; v.o_gs[a] = p2; v.o_gt[a] = p3; v.o_gq[a] = p4;
                v.o_gchi2[a] = p5; v.o_gndf[a] = 2 * nfit - 5; v.o_gnhits[a] = nfit; v.o_gsector[a] = v.o_sector[b_end];
                ph = 0;
            }
        }
    }
}

}  // namespace tpc
