// kf_refit.cuh -- refit of the output tracks over their final hit lists.
//
// One lane per track, as a small state machine that advances ONE pad row per loop trip (transport, and the
// update when the row holds the track's next hit), so that the 32 lanes of a warp stay on the same code whatever
// their tracks' lengths; a lane whose track is done takes the next track from a device counter at once.
// The hits of a track -- (y,z) and pad row, in hit-list order, written by K6c -- are read one ahead of their use.
// No search and no gate: every hit of the list is a measurement.  The arithmetic is fit_transport / fit_update of
// kf_kernels.cuh, i.e. what DESIGN.md "O5" parenthesises.
//   phase 1: up pass from the lowest hit (direction from the first two hits, q = 0, prior covariance)
//   phase 2: down pass = fresh fit at the top hit reached, (s, t, q) of the up pass
#pragma once
#include "common.cuh"
#include "kf_kernels.cuh"

namespace tpc {

constexpr int kRfThreads = 128;
constexpr int kRfBlocksPerSM = 6;

__global__ void __launch_bounds__(kRfThreads, kRfBlocksPerSM) k_refit(const View v, const __grid_constant__ Const c) {
    const int T = (int)v.cnt[CNT_TRACKS];
    const int lane = lane_id();
    unsigned long long* const cursor = &v.kf_cursor[2];
    Fit f;
    f.n = 0; f.chi2 = 0.f;
    float s_s = 0.f, s_t = 0.f, s_q = 0.f;          // sin phi, tg lambda, q/pT right after the last update (up pass)
    float ty = 0.f, tz = 0.f;                        // the hit of that update
    float uy = 0.f, uz = 0.f;                        // y, z of the up pass right after that update
    float p0 = 0.f, p1 = 0.f, p2 = 0.f, p3 = 0.f, p4 = 0.f, p5 = 0.f;   // down pass: state after its last update
    float ny = 0.f, nz = 0.f;                        // the track's next hit, read one trip ahead
    int nrow = -1;
    int ph = 0, ti = 0, h0 = 0, m = 0, k = 0, ktop = 0, row = 0, rfirst = 0, rlast = 0, rtop = 0, rref = 0, nfit = 0;
    unsigned visits = 0;
    bool more = true;
    for (;;) {
        const unsigned idle = __ballot_sync(kFull, ph == 0);
        if (idle && more) {
            int b = 0;
            if (lane == 0) b = (int)atomicAdd(cursor, (unsigned long long)__popc(idle));
            b = __shfl_sync(kFull, b, 0);
            if (b >= T) more = false;
            const int cand = b + __popc(idle & lanemask_lt());
            if (ph == 0 && cand < T && v.o_n_hits[cand] < 2) v.trk_rows[cand] = -1;
            if (ph == 0 && cand < T && v.o_n_hits[cand] >= 2) {
                ti = cand; h0 = v.trk_hit0[ti]; m = v.o_n_hits[ti];
                const float2 a0 = v.o_hit_yz[h0], a1 = v.o_hit_yz[h0 + 1];
                rfirst = v.o_hit_row[h0]; rlast = v.o_hit_row[h0 + m - 1];
                const int r1 = v.o_hit_row[h0 + 1];
                const float dx = c.row_x[r1] - c.row_x[rfirst];
                const float dy = a1.x - a0.x, dz = a1.y - a0.y;
                const float dl = sqrtf(dx * dx + dy * dy);
                f.y = a0.x; f.z = a0.y; f.s = dy / dl; f.t = dz / dl; f.q = 0.f;
                fit_prior(f, c); f.n = 1;
                s_s = f.s; s_t = f.t; s_q = f.q; ty = a0.x; tz = a0.y; uy = a0.x; uz = a0.y;
                row = rfirst; rtop = rfirst; ktop = 0; k = 1; ny = a1.x; nz = a1.y; nrow = r1;
                ph = 1;
            }
        }
        if (__all_sync(kFull, ph == 0)) break;
        const bool up = ph == 1;
        bool end = false, upd = false;
        if (ph != 0) {
            const int prev = row;
            row += up ? 1 : -1;
            end = up ? row > rlast : row < rfirst;
            if (!end) end = !fit_transport(f, c.row_x[prev], c.row_x[row], c);
            if (!end) { visits++; upd = row == nrow; }
        }
        __syncwarp();
        if (upd) {
            const float iwy = 1.f / (f.c00 + c.sigma_y2);
            fit_update(f, ny, nz, iwy, c);
            if (up) { s_s = f.s; s_t = f.t; s_q = f.q; ty = ny; tz = nz; uy = f.y; uz = f.z; rtop = row; ktop = k; k++; }
            else { p0 = f.y; p1 = f.z; p2 = f.s; p3 = f.t; p4 = f.q; p5 = f.chi2; rref = row; nfit = f.n; k--; }
            nrow = -1;
            if (k >= 0 && k < m) { const float2 hn = v.o_hit_yz[h0 + k]; ny = hn.x; nz = hn.y; nrow = v.o_hit_row[h0 + k]; }
        }
        __syncwarp();
        if (ph != 0 && end) {
            if (up) {   // outer state for O9, then a fresh fit at the top hit reached
                v.o_xo[ti] = c.row_x[rtop]; v.o_yo[ti] = uy; v.o_zo[ti] = uz; v.o_so[ti] = s_s; v.o_to[ti] = s_t; v.o_qo[ti] = s_q;
                f.y = ty; f.z = tz; f.s = s_s; f.t = s_t; f.q = s_q;
                fit_prior(f, c); f.n = 1;
                p0 = ty; p1 = tz; p2 = s_s; p3 = s_t; p4 = s_q; p5 = 0.f; rref = rtop; nfit = 1;
                row = rtop; k = ktop - 1;
                nrow = -1;
                if (k >= 0) { const float2 hn = v.o_hit_yz[h0 + k]; ny = hn.x; nz = hn.y; nrow = v.o_hit_row[h0 + k]; }
                ph = 2;
            } else {
                v.o_x[ti] = c.row_x[rref];
                v.o_y[ti] = p0; v.o_z[ti] = p1; v.o_sinphi[ti] = p2; v.o_tgl[ti] = p3; v.o_qpt[ti] = p4; v.o_chi2[ti] = p5;
                v.o_ndf[ti] = 2 * nfit - 5;
                v.trk_rows[ti] = rref | (rtop << 8);
                if (c.p.merge) atomicAdd(&v.dn_count[v.trk_task[ti] * c.n_rows + rref], 1);   // O9: lists by (task, first row)
                ph = 0;
            }
        }
    }
    unsigned long long vs = visits;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) vs += __shfl_xor_sync(kFull, vs, o);
    if (lane == 0 && vs) atomicAdd(&v.cnt[CNT_REFIT_VISITS], vs);
}

}  // namespace tpc
