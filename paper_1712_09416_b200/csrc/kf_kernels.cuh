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
    const float adl = sqrtf(dl2);
    const float dl = (dx < 0.f) ? -adl : adl;
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

// two scalar updates, y then z; iwy = 1 / (C_yy + sigma_y^2) of the predicted state
__device__ __forceinline__ void fit_update(Fit& f, float my, float mz, float iwy, const Const& c) {
    {
        const float r = my - f.y;
        const float w = iwy;
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

// selection key of tracklet i: more hits first, then the lower canonical id within the sector task
__device__ __forceinline__ uint32_t tl_key(const View& v, int i, int nh, int task_bin0) {
    const int id_in_task = i - v.seed_start[task_bin0];
    return ((uint32_t)nh << 24) | (uint32_t)(0xffffff - id_in_task);
}

// ---------------------------------------------------------------------------------------------------------
// K5 tracklet constructor.  Persistent CTAs; every lane runs one tracklet as a small state machine that
// advances ONE pad row per loop trip (transport -> candidate -> update), so that the 32 lanes of a warp stay
// on the same code whatever their tracklets' lengths; a lane whose tracklet is finished takes the next start
// hit from a device counter at once.
//   phase 1: up pass, following the cleaned links      phase 2: up pass, extending by search
//   phase 3: down pass = fresh fit from the top hit through everything recorded, searching the empty rows
// Window search: the candidates of one grid row of the window are contiguous in memory and
// are loaded kKfUnroll at a time; the best hit = min gate value, exact ties -> lowest caller's index, whatever the
// order of evaluation.  The warp is brought together (__syncwarp) before the transport, the search and the update,
// so that each runs once per trip for all lanes that need it.
// The row -> hit table of a tracklet ([tracklet][row], row-local 16-bit hit numbers) is written as the passes
// go; when a tracklet ends, its warp claims the hits of rows first..last for the selector (K6a: atomicMax of the
// tracklet's key on owner[hit]).
// ---------------------------------------------------------------------------------------------------------
constexpr int kKfThreads = 128;
#ifndef TPC_KF_BLOCKS
#define TPC_KF_BLOCKS 6
#endif
#ifndef TPC_KF_SWEEP
#define TPC_KF_SWEEP 1
#endif
#ifndef TPC_KF_SCHED
#define TPC_KF_SCHED 1
#endif
#ifndef TPC_KF_UNROLL
#define TPC_KF_UNROLL 2
#endif
constexpr int kKfBlocksPerSM = TPC_KF_BLOCKS;
constexpr int kKfUnroll = TPC_KF_UNROLL;       // candidates of a grid row loaded at once

__global__ void __launch_bounds__(kKfThreads, kKfBlocksPerSM) k_construct(const View v, const __grid_constant__ Const c) {
    const int S = min(v.seed_start[v.n_bins], v.S_cap);
    const int nr = c.n_rows, D = c.p.link_step;
    const int lane = lane_id();
    unsigned long long* const cursor = v.kf_cursor;   // start hits taken from each share of the list
    unsigned sm = 0, n_sm_u;
    asm("mov.u32 %0, %%smid;" : "=r"(sm));
    asm("mov.u32 %0, %%nsmid;" : "=r"(n_sm_u));
    const int n_sm = (int)n_sm_u;
    int victim = 0;   // SMs whose share this warp has found exhausted, starting with its own

    Fit f;
    float p0 = 0.f, p1 = 0.f, p2 = 0.f, p3 = 0.f, p4 = 0.f, p5 = 0.f;  // up: top hit (y,z), s,t,q there; down: result
    float cy = 0.f, cz = 0.f;    // coordinates of the hit the up pass follows next
    int ph = 0;                  // 0 idle, 1 up/follow, 2 up/extend, 3 down
    int i = 0, row = 0, r0 = 0, top = 0, first = 0, nh = 0, tb = 0, cur = -1, rcur = 0, miss = 0;
    uint16_t enext = kNoHit;     // down pass: table entry of the row below, loaded one trip ahead
    f.n = 0;
    unsigned visits = 0, claimed = 0;
    bool more = true;

    for (;;) {
        // ---- idle lanes take the next start hits: first from this SM's share of the list, then from the others' ----
        const unsigned idle = __ballot_sync(kFull, ph == 0);
        if (idle && more) {
            int b = 0, e = 0;
            if (lane == 0) {
                const int want = __popc(idle);
#if TPC_KF_SCHED == 1
                // one cursor for the whole list: all SMs work in the same narrow window of start hits
                const int got = (int)atomicAdd(&cursor[0], (unsigned long long)want);
                if (got < S) { b = got; e = S; } else victim = n_sm;
#elif TPC_KF_SCHED == 2
                // event by event: an SM takes its own share of every event first (the SMs then stay in the same
                // one or two events, whose hits fit the L2), and only then the other SMs' shares
                const int ne = v.n_events, bpe = c.n_sectors * nr;
                while (victim < n_sm * ne) {
                    const int vs = victim / ne, ev = victim - vs * ne;
                    const int s = (sm + vs) % n_sm;
                    const int e_lo = min(v.seed_start[ev * bpe], S), e_n = min(v.seed_start[(ev + 1) * bpe], S) - e_lo;
                    const int lo = e_lo + (int)((long long)e_n * s / n_sm), hi = e_lo + (int)((long long)e_n * (s + 1) / n_sm);
                    const int got = lo + (int)atomicAdd(&cursor[ev * n_sm + s], (unsigned long long)want);
                    if (got < hi) { b = got; e = hi; break; }
                    victim++;
                }
#else
                while (victim < n_sm) {
                    const int s = (sm + victim) % n_sm;
                    const int lo = (int)((long long)S * s / n_sm), hi = (int)((long long)S * (s + 1) / n_sm);
                    const int got = lo + (int)atomicAdd(&cursor[s], (unsigned long long)want);
                    if (got < hi) { b = got; e = hi; break; }
                    victim++;
                }
#endif
            }
            b = __shfl_sync(kFull, b, 0); e = __shfl_sync(kFull, e, 0); victim = __shfl_sync(kFull, victim, 0);
            if (victim >= n_sm * (TPC_KF_SCHED == 2 ? v.n_events : 1)) more = false;
            const int cand = b + __popc(idle & lanemask_lt());
            if (ph == 0 && cand < e) {
                i = cand;
                const int h0 = v.seeds[i];
                const int bin0 = v.seed_bin[i];
                r0 = bin0 % nr; tb = bin0 - r0;
                const int h1 = v.clink_up[h0];
                const float2 a0 = v.shit[h0], a1 = v.shit[h1];
                const int base0 = load_desc_n(v, bin0).x;
                const float dx = c.row_x[r0 + D] - c.row_x[r0];
                const float dy = a1.x - a0.x, dz = a1.y - a0.y;
                const float dl = sqrtf(dx * dx + dy * dy);
                f.y = a0.x; f.z = a0.y; f.s = dy / dl; f.t = dz / dl; f.q = 0.f;
                fit_prior(f, c); f.n = 1;
                v.tl_tab[(size_t)i * v.tab_stride + r0] = (uint16_t)(h0 - base0);
                p0 = a0.x; p1 = a0.y; p2 = f.s; p3 = f.t; p4 = f.q;
                top = r0; row = r0; cur = h1; rcur = r0 + D; cy = a1.x; cz = a1.y; miss = 0;
                ph = 1;
            }
        }
        if (__all_sync(kFull, ph == 0)) break;

        // ---- one pad row, part 1: transport and the candidate that is already known ----
        const bool active = ph != 0;
        const bool up = ph != 3;
        uint16_t* const gt = v.tl_tab + (size_t)i * v.tab_stride;
        bool end = false, search = false, counted = false;   // counted: the edge test and the gap count apply
        int acc = -1;
        float ay = 0.f, az = 0.f, iwy = 0.f, iwz = 0.f;
        int4 dn = make_int4(0, 0, 1, 1);
        if (active) {
            const int prev = row;
            row += up ? 1 : -1;
            end = up ? (row >= nr) : (row < 0);
            if (!end) {
                // loads that do not depend on the fit are issued before the transport
                dn = load_desc_n(v, tb + row);
                int nxt = -1, known = -1;
                float ky = 0.f, kz = 0.f;
                if (ph == 1) {
                    if (row == rcur) { known = cur; ky = cy; kz = cz; nxt = v.clink_up[cur]; }
                } else if (ph == 3 && row >= r0) {
                    const uint16_t e = enext;
                    if (row > r0) enext = gt[row - 1];
                    if (e != kNoHit) { known = dn.x + e; const float2 hk = v.shit[known]; ky = hk.x; kz = hk.y; }
                }
                end = !fit_transport(f, c.row_x[prev], c.row_x[row], c);
                if (!end) {
                    visits++;
                    iwy = 1.f / (f.c00 + c.sigma_y2); iwz = 1.f / (f.c11 + c.sigma_z2);
                    bool gate_ok = false;
                    if (known >= 0) {   // the gate value of (ky, kz) on the predicted state
                        const float ry = ky - f.y, rz = kz - f.z;
                        gate_ok = (ry * ry) * iwy + (rz * rz) * iwz <= c.p.chi2_link;
                        if (gate_ok) { acc = known; ay = ky; az = kz; }
                    }
                    if (ph == 1) {
                        if (row == rcur) {
                            if (gate_ok) {
                                cur = nxt; rcur += D;
                                if (cur < 0) ph = 2;
                                else { const float2 hn = v.shit[cur]; cy = hn.x; cz = hn.y; }
                            } else { ph = 2; search = true; counted = true; }
                        }   // else: in-between row of a step-2 link
                    } else if (ph == 2) {
                        search = true; counted = true;
                    } else {
                        search = row < r0 || known < 0;
                        counted = row < r0;
                    }
                    if (search && counted && fabsf(f.y) > c.row_x[row] * c.tan_half_angle + c.p.edge_margin) {
                        end = true; search = false;
                    }
                }
            }
        }

        // ---- part 2: the window searches of this trip ----
        __syncwarp();
        if (search && dn.y > 0) {
            const float wy = fminf(fmaxf(c.p.win_nsigma * sqrtf(f.c00 + c.sigma_y2), c.p.win_min), c.p.win_max);
            const float wz = fminf(fmaxf(c.p.win_nsigma * sqrtf(f.c11 + c.sigma_z2), c.p.win_min), c.p.win_max);
            const float4 gf = load_desc_f(v, tb + row);
            const CellWin w = cell_window(gf, dn.z, dn.w, f.y, f.z, wy, wz);
            const uint16_t* cs = cell_table(v, tb + row, dn.x);
            const float2* hits = v.shit + dn.x;
            float bg = 0.f;
            int bp = -1;
            for (int iz = w.iz0; iz <= w.iz1; iz++) {
                int p = __ldg(&cs[iz * dn.z + w.iy0]);
                const int pe = __ldg(&cs[iz * dn.z + w.iy1 + 1]);
                for (; p < pe; p += kKfUnroll) {   // the candidates of a grid row are contiguous: loads go out together
                    float2 h[kKfUnroll];
#pragma unroll
                    for (int k = 0; k < kKfUnroll; k++) h[k] = __ldg(&hits[min(p + k, pe - 1)]);
#pragma unroll
                    for (int k = 0; k < kKfUnroll; k++) {
                        const float ry = h[k].x - f.y, rz = h[k].y - f.z;
                        if (p + k < pe && fabsf(ry) <= wy && fabsf(rz) <= wz) {
                            const float gv = (ry * ry) * iwy + (rz * rz) * iwz;   // the gate value of h[k]
                            bool take = bp < 0 || gv < bg;
                            if (!take && gv == bg) take = v.sorig[dn.x + p + k] < v.sorig[dn.x + bp];
                            if (take) { bg = gv; bp = p + k; ay = h[k].x; az = h[k].y; }
                        }
                    }
                }
            }
            if (bp >= 0 && bg <= c.p.chi2_ext) acc = dn.x + bp;
        }
        __syncwarp();

        // ---- part 3: bookkeeping, update, end of a pass (the warp is brought together before each piece) ----
        bool finished = false, upd = false;
        if (active) {
            if (search) {
                if (acc >= 0) miss = 0;
                else if (counted && ++miss > c.p.max_gap) end = true;
            }
            if (!end) {
                gt[row] = acc >= 0 ? (uint16_t)(acc - dn.x) : kNoHit;
                upd = acc >= 0;
            }
        }
        __syncwarp();
        if (upd) {
            fit_update(f, ay, az, iwy, c);
            p0 = up ? ay : f.y; p1 = up ? az : f.z; p2 = f.s; p3 = f.t; p4 = f.q; p5 = f.chi2;
            top = up ? row : top; first = row; nh = f.n;
        }
        __syncwarp();
        if (active && end) {
            if (up) {   // start the down pass at the top hit
                f.y = p0; f.z = p1; f.s = p2; f.t = p3; f.q = p4;
                fit_prior(f, c); f.n = 1;
                p5 = 0.f;
                row = top; first = top; nh = 1; miss = 0;
                enext = top > r0 ? gt[top - 1] : kNoHit;
                ph = 3;
            } else {
                finished = true;
            }
        }

        // ---- finished tracklets: parameters, claim of the hits of rows first..top (K6a) ----
        unsigned fin = __ballot_sync(kFull, finished);
        if (fin) {
            uint32_t key = 0;
            if (finished) {
                v.tl_rows[i] = first | (top << 8) | (nh << 16);
                const int sc = v.S_cap;
                v.tl_par[i] = p0; v.tl_par[sc + i] = p1; v.tl_par[2 * sc + i] = p2; v.tl_par[3 * sc + i] = p3;
                v.tl_par[4 * sc + i] = p4; v.tl_par[5 * sc + i] = p5;
                if (nh >= c.p.min_tracklet_hits) key = tl_key(v, i, nh, tb);
                ph = 0;
            }
            fin = __ballot_sync(kFull, key != 0);
            __syncwarp();
            while (fin) {
                const int L = __ffs(fin) - 1;
                fin &= fin - 1;
                const int li = __shfl_sync(kFull, i, L), lfirst = __shfl_sync(kFull, first, L);
                const int ltop = __shfl_sync(kFull, top, L), ltb = __shfl_sync(kFull, tb, L);
                const uint32_t lkey = __shfl_sync(kFull, key, L);
                const uint16_t* lt = v.tl_tab + (size_t)li * v.tab_stride;
                for (int r = lfirst + lane; r <= ltop; r += 32) {
                    const uint16_t e = lt[r];
                    if (e != kNoHit) {
                        atomicMax(&v.owner[load_desc_n(v, ltb + r).x + e], lkey);
                        claimed++;
                    }
                }
            }
        }
    }
    unsigned long long vs = visits, cl = claimed;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { vs += __shfl_xor_sync(kFull, vs, o); cl += __shfl_xor_sync(kFull, cl, o); }
    if (lane == 0) {
        if (vs) atomicAdd(&v.cnt[CNT_ROW_VISITS], vs);
        if (cl) atomicAdd(&v.cnt[CNT_TL_HITS], cl);
    }
}

// ---------------------------------------------------------------------------------------------------------
// K6 selector.  key = n_hits << 24 | (2^24 - 1 - id within the task): larger = more hits, then lower
// canonical id.  owner[hit] = max key over tracklets (n_hits >= min_tracklet_hits) holding the hit (claimed by
// K5 as each tracklet ends).  One warp per tracklet, lanes over its rows: coalesced table reads.
// ---------------------------------------------------------------------------------------------------------
constexpr int kSelThreads = 128;

// K6b: hits each tracklet owns; a track is kept when it owns at least min_track_hits
__global__ void __launch_bounds__(kSelThreads) k_count_owned(const View v, const __grid_constant__ Const c) {
    const int S = min(v.seed_start[v.n_bins], v.S_cap);
    const int nr = c.n_rows;
    const int lane = lane_id();
    for (int i = (blockIdx.x * kSelThreads + threadIdx.x) >> 5; i < S; i += (gridDim.x * kSelThreads) >> 5) {
    const int pk = v.tl_rows[i];
    const int nh = pk >> 16;
    int own = 0;
    if (nh >= c.p.min_tracklet_hits) {
        const int first = pk & 0xff, last = (pk >> 8) & 0xff;
        const int bin = v.seed_bin[i];
        const int tb = bin - bin % nr;
        const uint32_t key = tl_key(v, i, nh, tb);
        const uint16_t* gt = v.tl_tab + (size_t)i * v.tab_stride;
        for (int r = first + lane; r <= last; r += 32) {
            const uint16_t e = gt[r];
            if (e != kNoHit && v.owner[load_desc_n(v, tb + r).x + e] == key) own++;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) own += __shfl_xor_sync(kFull, own, o);
    }
    if (lane == 0) {
        const int keep = own >= c.p.min_track_hits;
        v.tl_keep[i] = keep;
        v.tl_nown[i] = keep ? own : 0;
    }
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

// K6c: output tracks in canonical order; hit lists row-ascending (ballot + prefix popcount keeps the order)
__global__ void __launch_bounds__(kSelThreads) k_write_tracks(const View v, const __grid_constant__ Const c) {
    const int S = min(v.seed_start[v.n_bins], v.S_cap);
    const int nr = c.n_rows;
    const int lane = lane_id();
    for (int i = (blockIdx.x * kSelThreads + threadIdx.x) >> 5; i < S; i += (gridDim.x * kSelThreads) >> 5) {
    if (!v.tl_keep[i]) continue;
    const int pk = v.tl_rows[i];
    const int nh = pk >> 16, first = pk & 0xff, last = (pk >> 8) & 0xff;
    const int bin = v.seed_bin[i];
    const int tb = bin - bin % nr;
    const uint32_t key = tl_key(v, i, nh, tb);
    int ho = v.hit_scan[i];
    if (lane == 0) {
        const int ti = v.trk_scan[i];
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
    const uint16_t* gt = v.tl_tab + (size_t)i * v.tab_stride;
    for (int r0 = first; r0 <= last; r0 += 32) {
        const int r = r0 + lane;
        int h = -1;
        if (r <= last) {
            const uint16_t e = gt[r];
            if (e != kNoHit) { h = load_desc_n(v, tb + r).x + e; if (v.owner[h] != key) h = -1; }
        }
        const unsigned m = __ballot_sync(kFull, h >= 0);
        if (h >= 0) v.o_hit_idx[ho + __popc(m & lanemask_lt())] = v.sorig[h];
        ho += __popc(m);
    }
    }
}

}  // namespace tpc
