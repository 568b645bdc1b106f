// kf_sweep.cuh -- K5 tracklet constructor as row sweeps with the pad-row data staged in shared memory by TMA.
//
// One CTA works on one sector task (or on a fixed share of its start hits) and sweeps the pad rows in order: upwards
// for the up passes (k_sweep<true>), downwards for the down passes (k_sweep<false>).  A producer warp streams the
// rows -- hits and grid cell table of row r, one cp.async.bulk each, completion on an mbarrier -- through a ring of
// kSwSlots shared-memory slots; the consumer warps hold one tracklet per lane and advance all of them by the row
// that has just arrived: transport, candidate (linked / recorded hit, or window search in the staged row), update.
// A lane whose tracklet has ended takes, at the next row, a start hit of THAT row (the start-hit list is ordered by
// row), so the lanes stay filled while the sweep goes on; what a sweep could not take is left for the next sweep of
// the same CTA.  Everything a step reads -- descriptors, hits, cell table -- is in shared memory; global memory
// sees the bulk row copies, the row -> hit table and one record per tracklet.
//
// The up pass parks (top row, top hit, sin phi, tg lambda, q/pT there) per tracklet; k_dn_scatter buckets these
// records by (task, top row); the down sweep picks them up at their top row.  The arithmetic is that of
// kf_kernels.cuh (fit_transport / fit_update), so every decision is the one DESIGN.md "O5" describes.
#pragma once
#include "common.cuh"
#include "kf_kernels.cuh"

namespace tpc {

#ifndef TPC_SW_WARPS
#define TPC_SW_WARPS 6
#endif
#ifndef TPC_SW_BLOCKS
#define TPC_SW_BLOCKS 4
#endif
#ifndef TPC_SW_PSLEEP
#define TPC_SW_PSLEEP 500
#endif
#ifndef TPC_SW_CSLEEP
#define TPC_SW_CSLEEP 100
#endif
#ifndef TPC_SW_SLOTS
#define TPC_SW_SLOTS 2
#endif
constexpr int kSwWarps = TPC_SW_WARPS;                 // consumer warps of a CTA (one more warp produces)
constexpr int kSwThreads = (kSwWarps + 1) * 32;
constexpr int kSwBlocksPerSM = TPC_SW_BLOCKS;
constexpr int kSwSlots = TPC_SW_SLOTS;                 // rows in flight
constexpr int kSwCap = 640;                            // hits of a row staged in shared memory; larger rows are read in place
constexpr int kSwHitBytes = (kSwCap + 2) * 8;          // + alignment slack of the bulk copy (16-byte granules)
constexpr int kSwCellEntries = kCellsPerHit * kSwCap + kCellPad + 16;
constexpr int kSwCellBytes = kSwCellEntries * 2;
static_assert(kSwHitBytes % 16 == 0 && kSwCellBytes % 16 == 0, "bulk copies are 16-byte granular");
constexpr unsigned kSwSpinMax = 1u << 22;              // bounded waits: a lost signal ends the kernel with kErrHang

struct __align__(16) SeedRec { float y0, z0, y1, z1; int32_t h0, h1, pad0, pad1; };   // start hit, its up-link
struct __align__(16) UpRec { float y, z, s, t, q; int32_t r0, top, id; };             // what the up pass hands down

struct __align__(128) SweepSmem {
    BinDesc desc[TPC_MAX_ROWS + 1];                    // the task's row descriptors
    unsigned char hits[kSwSlots][kSwHitBytes];
    unsigned char cells[kSwSlots][kSwCellBytes];
    int32_t lo[TPC_MAX_ROWS + 1];                      // first list entry of each row (start hits / parked tracklets)
    int32_t own[TPC_MAX_ROWS + 1];                     // entries of the row that are this CTA's to take
    int32_t next[TPC_MAX_ROWS + 1];                    // taken so far
    unsigned long long full[kSwSlots], empty[kSwSlots], tbar;
    int32_t cmd[kSwSlots];                             // row held by the slot; -1 = no more work
    int32_t task, k, abort;
};

// ---- mbarrier / bulk-copy wrappers (PTX ISA: mbarrier, cp.async.bulk) ----
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* b, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* b) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned long long* b, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(unsigned long long* b, uint32_t parity) {
    uint32_t ok;
    asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                 : "=r"(ok) : "r"(smem_u32(b)), "r"(parity) : "memory");
    return ok != 0;
}
#ifndef TPC_SW_WAITMODE
#define TPC_SW_WAITMODE 1
#endif
// try_wait that lets the hardware suspend the warp for up to `ns` before it answers
__device__ __forceinline__ bool mbar_try_wait_hint(unsigned long long* b, uint32_t parity, uint32_t ns) {
    uint32_t ok;
    asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n selp.u32 %0, 1, 0, p;\n}"
                 : "=r"(ok) : "r"(smem_u32(b)), "r"(parity), "r"(ns) : "memory");
    return ok != 0;
}
template <int SLEEP_NS>
__device__ __forceinline__ bool mbar_wait(unsigned long long* b, uint32_t parity, volatile int32_t* abort) {
    if (mbar_try_wait(b, parity)) return true;
#if TPC_SW_WAITMODE == 1
    // suspended waits: a waiting warp issues nothing until the phase completes or the hint runs out
    for (unsigned n = 0; n < (1u << 17); n++) {
        if (mbar_try_wait_hint(b, parity, 20000u)) return true;
        if ((n & 63u) == 63u && *abort) return false;
    }
#else
    for (unsigned n = 0; n < kSwSpinMax; n++) {   // back off: a spinning warp takes issue slots from the working ones
        __nanosleep(SLEEP_NS);
        if (mbar_try_wait(b, parity)) return true;
        if ((n & 255u) == 255u && *abort) return false;
    }
#endif
    *abort = 1;
    return false;
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, unsigned long long* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// where row `row` of task `tb / nr` sits in a slot (the bulk copy starts at the 16-byte boundary below the data)
__device__ __forceinline__ size_t cell_index(int base, int bin) { return (size_t)kCellsPerHit * base + (size_t)bin * kCellPad; }

// ---------------------------------------------------------------------------------------------------------
// producer warp: hands the CTA its units of work and streams their rows
// ---------------------------------------------------------------------------------------------------------
template <bool UP>
__device__ __forceinline__ void sweep_producer(const View& v, const Const& c, SweepSmem& sm) {
    const int lane = lane_id();
    const int nr = c.n_rows, K = v.kf_K, n_units = v.n_tasks * K;
    const int32_t* lst = UP ? v.seed_start : v.dn_start;
    volatile int32_t* const abort = &sm.abort;
    uint32_t it = 0, tphase = 0;
    bool ok = true;
    while (ok) {
        int u = 0;
        if (lane == 0) u = (int)atomicAdd(&v.kf_cursor[UP ? 0 : 1], 1ull);
        u = __shfl_sync(kFull, u, 0);
        if (u >= n_units) break;
        const int task = u / K, k = u - task * K, tb = task * nr;
        // the consumers are idle here (start of the kernel, or all slots drained): the task's tables may be replaced
        if (lane == 0) {
            mbar_arrive_expect_tx(&sm.tbar, (uint32_t)nr * 32u);
            bulk_g2s(sm.desc, v.desc + tb, (uint32_t)nr * 32u, &sm.tbar);
            sm.task = task; sm.k = k;
        }
        for (int r = lane; r < nr; r += 32) {
            const int lo = lst[tb + r], n = lst[tb + r + 1] - lo;
            sm.lo[r] = lo; sm.own[r] = n > k ? (n - k + K - 1) / K : 0; sm.next[r] = 0;
        }
        if (lane == 0) ok = mbar_wait<100>(&sm.tbar, tphase, abort);
        tphase ^= 1u;
        ok = __shfl_sync(kFull, (int)ok, 0) != 0;
        __syncwarp();
        while (ok) {   // sweeps, until nothing of this CTA's share is left
            int f = UP ? nr : -1;
            for (int r = lane; r < nr; r += 32)
                if (*(volatile int32_t*)&sm.next[r] < sm.own[r]) f = UP ? min(f, r) : max(f, r);
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                const int g = __shfl_xor_sync(kFull, f, o);
                f = UP ? min(f, g) : max(f, g);
            }
            if (UP ? f >= nr : f < 0) break;
            if (lane == 0) {
                for (int row = f; UP ? row < nr : row >= 0; row += UP ? 1 : -1) {
                    const int s = (int)(it % kSwSlots);
                    if (!(ok = mbar_wait<TPC_SW_PSLEEP>(&sm.empty[s], ((it / kSwSlots) & 1u) ^ 1u, abort))) break;
                    sm.cmd[s] = row;
                    const BinDesc& d = sm.desc[row];
                    if (d.n > 0 && d.n <= kSwCap) {
                        const int offh = d.base & 1;
                        const uint32_t hb = (uint32_t)((offh + d.n + 1) & ~1) * 8u;
                        const size_t g = cell_index(d.base, tb + row);
                        const int offc = (int)(g & 7);
                        const uint32_t cb = ((uint32_t)(offc + d.ny * d.nz + 1) * 2u + 15u) & ~15u;
                        mbar_arrive_expect_tx(&sm.full[s], hb + cb);
                        bulk_g2s(sm.hits[s], v.shit + (d.base - offh), hb, &sm.full[s]);
                        bulk_g2s(sm.cells[s], v.cells + (g - offc), cb, &sm.full[s]);
                    } else {
                        mbar_arrive(&sm.full[s]);
                    }
                    it++;
                }
                // drain: the consumers must be through with the sweep before its leftovers are counted
                for (uint32_t j = it > (uint32_t)kSwSlots ? it - kSwSlots : 0; ok && j < it; j++)
                    ok = mbar_wait<TPC_SW_PSLEEP>(&sm.empty[j % kSwSlots], (j / kSwSlots) & 1u, abort);
            }
            it = __shfl_sync(kFull, it, 0);
            ok = __shfl_sync(kFull, (int)ok, 0) != 0;
            __syncwarp();
        }
    }
    if (lane == 0) {
        const int s = (int)(it % kSwSlots);
        if (ok) ok = mbar_wait<TPC_SW_PSLEEP>(&sm.empty[s], ((it / kSwSlots) & 1u) ^ 1u, abort);
        sm.cmd[s] = -1;
        mbar_arrive(&sm.full[s]);
        if (!ok) atomicOr((unsigned int*)&v.cnt[CNT_ERR], kErrHang);
    }
}

// ---------------------------------------------------------------------------------------------------------
// window search in one row: min gate value, exact ties -> lowest caller's index
// hits / cs point to the row's hits and cell table (shared memory, or global for an oversized row)
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ int sweep_search(const View& v, const Const& c, const Fit& f, const float4& gf, const int4& dn,
                                            const float2* hits, const uint16_t* cs, float iwy, float iwz, float& ay,
                                            float& az, float& bg) {
    const float wy = fminf(fmaxf(c.p.win_nsigma * sqrtf(f.c00 + c.sigma_y2), c.p.win_min), c.p.win_max);
    const float wz = fminf(fmaxf(c.p.win_nsigma * sqrtf(f.c11 + c.sigma_z2), c.p.win_min), c.p.win_max);
    const CellWin w = cell_window(gf, dn.z, dn.w, f.y, f.z, wy, wz);
    int bp = -1;
    bg = __int_as_float(0x7f800000);   // +inf: the first hit inside the window always wins
    for (int iz = w.iz0; iz <= w.iz1; iz++) {
        int p = cs[iz * dn.z + w.iy0];
        const int pe = cs[iz * dn.z + w.iy1 + 1];
        for (; p < pe; p++) {
            const float2 h = hits[p];
            const float ry = h.x - f.y, rz = h.y - f.z;
            if (fabsf(ry) <= wy && fabsf(rz) <= wz) {
                const float gv = (ry * ry) * iwy + (rz * rz) * iwz;   // the gate value of h
                bool take = gv < bg;
                if (gv == bg) take = v.sorig[dn.x + p] < v.sorig[dn.x + bp];   // exact tie (gv is finite: bp >= 0 here)
                if (take) { bg = gv; bp = p; }
            }
        }
    }
    if (bp >= 0) { const float2 h = hits[bp]; ay = h.x; az = h.y; }
    return bp;
}

// ---------------------------------------------------------------------------------------------------------
// K5: up sweep (UP) / down sweep (!UP)
// ---------------------------------------------------------------------------------------------------------
template <bool UP>
__global__ void __launch_bounds__(kSwThreads, kSwBlocksPerSM) k_sweep(const View v, const __grid_constant__ Const c) {
    __shared__ SweepSmem sm;
    const int warp = threadIdx.x >> 5, lane = lane_id();
    if (threadIdx.x == 0) {
        for (int s = 0; s < kSwSlots; s++) { mbar_init(&sm.full[s], 1); mbar_init(&sm.empty[s], kSwWarps); }
        mbar_init(&sm.tbar, 1);
        sm.abort = 0;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (warp == kSwWarps) { sweep_producer<UP>(v, c, sm); return; }

    const int nr = c.n_rows, D = c.p.link_step, K = v.kf_K;
    const int S = min(v.seed_start[v.n_bins], v.S_cap);
    volatile int32_t* const abort = &sm.abort;
    Fit f;
    float p0 = 0.f, p1 = 0.f, p2 = 0.f, p3 = 0.f, p4 = 0.f, p5 = 0.f;   // state right after the last accepted update
    int ph = 0;                  // 0 idle, 1 up/follow, 2 up/extend, 3 down
    int i = 0, r0 = 0, top = 0, first = 0, nh = 0, cur = -1, rcur = 0, miss = 0;
    uint16_t enext = kNoHit;     // down pass: table entry of the row below, loaded one step ahead
    f.n = 0; f.chi2 = 0.f;
    unsigned visits = 0, updates = 0;
    uint32_t it = 0;

    for (;;) {
        const int s = (int)(it % kSwSlots);
        if (!mbar_wait<TPC_SW_CSLEEP>(&sm.full[s], (it / kSwSlots) & 1u, abort)) break;
        const int row = sm.cmd[s];
        if (row < 0) break;
        const int tb = sm.task * nr;
        const BinDesc& dsc = sm.desc[row];
        const int4 dn = make_int4(dsc.base, dsc.n, dsc.ny, dsc.nz);
        const bool staged = dn.y <= kSwCap;
        const size_t cg = cell_index(dn.x, tb + row);
        const float2* const hits = staged ? reinterpret_cast<const float2*>(sm.hits[s]) + (dn.x & 1) : v.shit + dn.x;
        const uint16_t* const cs = staged ? reinterpret_cast<const uint16_t*>(sm.cells[s]) + (cg & 7) : v.cells + cg;

        // ---- idle lanes take what starts at this row ----
        bool started = false;
        const unsigned idle = __ballot_sync(kFull, ph == 0);
        if (idle && *(volatile int32_t*)&sm.next[row] < sm.own[row]) {
            int a = 0;
            if (lane == 0) a = atomicAdd(&sm.next[row], __popc(idle));
            a = __shfl_sync(kFull, a, 0);
            const int pos = a + __popc(idle & lanemask_lt());
            if (ph == 0 && pos < sm.own[row]) {
                const int e = sm.lo[row] + sm.k + K * pos;
                if (UP) {
                    if (e < S) {
                        const float4 a4 = __ldg(reinterpret_cast<const float4*>(&v.seed_rec[e]));
                        const int2 h01 = __ldg(reinterpret_cast<const int2*>(&v.seed_rec[e]) + 2);
                        i = e; r0 = row;
                        const float dx = c.row_x[r0 + D] - c.row_x[r0];
                        const float dy = a4.z - a4.x, dz = a4.w - a4.y;
                        const float dl = sqrtf(dx * dx + dy * dy);
                        f.y = a4.x; f.z = a4.y; f.s = dy / dl; f.t = dz / dl; f.q = 0.f;
                        fit_prior(f, c);
                        v.tl_tab[(size_t)i * v.tab_stride + r0] = (uint16_t)(h01.x - dn.x);
                        p0 = a4.x; p1 = a4.y; p2 = f.s; p3 = f.t; p4 = f.q;
                        top = r0; cur = h01.y; rcur = r0 + D; miss = 0;
                        ph = 1; started = true;
                    }
                } else {
                    const float4 a4 = __ldg(reinterpret_cast<const float4*>(&v.dn_rec[e]));
                    const float4 b4 = __ldg(reinterpret_cast<const float4*>(&v.dn_rec[e]) + 1);
                    p0 = a4.x; p1 = a4.y; p2 = a4.z; p3 = a4.w; p4 = b4.x; p5 = 0.f;
                    r0 = __float_as_int(b4.y); top = row; i = __float_as_int(b4.w);
                    f.y = p0; f.z = p1; f.s = p2; f.t = p3; f.q = p4;
                    fit_prior(f, c); f.n = 1;
                    first = top; nh = 1; miss = 0;
                    enext = top > r0 ? v.tl_tab[(size_t)i * v.tab_stride + top - 1] : kNoHit;
                    ph = 3; started = true;
                }
            }
        }

        // ---- one pad row for the tracklets under way, part 1: transport and the candidate that is already known ----
        const bool active = ph != 0 && !started;
        uint16_t* const gt = v.tl_tab + (size_t)i * v.tab_stride;
        bool end = false, search = false, counted = false;
        int acc = -1;
        uint16_t eold = kNoHit;
        float ay = 0.f, az = 0.f, iwy = 0.f, iwz = 0.f;
        if (active) {
            int nxt = -1, known = -1;
            float ky = 0.f, kz = 0.f;
            if (UP) {
                if (ph == 1 && row == rcur) { known = cur; nxt = __ldg(&v.clink_up[cur]); const float2 hk = hits[cur - dn.x]; ky = hk.x; kz = hk.y; }
            } else if (row >= r0) {
                eold = enext;
                if (row > r0) enext = gt[row - 1];
                if (eold != kNoHit) { known = dn.x + eold; const float2 hk = hits[eold]; ky = hk.x; kz = hk.y; }
            }
            end = !fit_transport(f, c.row_x[UP ? row - 1 : row + 1], c.row_x[row], c);
            if (!end) {
                visits++;
                iwy = 1.f / (f.c00 + c.sigma_y2); iwz = 1.f / (f.c11 + c.sigma_z2);
                bool gate_ok = false;
                if (known >= 0) {   // the gate value of (ky, kz) on the predicted state
                    const float ry = ky - f.y, rz = kz - f.z;
                    gate_ok = (ry * ry) * iwy + (rz * rz) * iwz <= c.p.chi2_link;
                    if (gate_ok) { acc = known; ay = ky; az = kz; }
                }
                if (UP) {
                    if (ph == 1) {
                        if (row == rcur) {
                            if (gate_ok) { cur = nxt; rcur += D; if (cur < 0) ph = 2; }
                            else { ph = 2; search = true; counted = true; }
                        }   // else: in-between row of a step-2 link
                    } else {
                        search = true; counted = true;
                    }
                } else {
                    search = row < r0 || known < 0;
                    counted = row < r0;
                }
                if (search && counted && fabsf(f.y) > c.row_x[row] * c.tan_half_angle + c.p.edge_margin) {
                    end = true; search = false;
                }
            }
        }

        // ---- part 2: the window searches of this row ----
        __syncwarp();
        if (search && dn.y > 0) {
            const float4 gf = make_float4(dsc.y0, dsc.z0, dsc.idy, dsc.idz);
            float bg = 0.f;   // a lane that searches has accepted nothing yet on this row: (ay, az) are free
            const int bp = sweep_search(v, c, f, gf, dn, hits, cs, iwy, iwz, ay, az, bg);
            if (bp >= 0 && bg <= c.p.chi2_ext) acc = dn.x + bp;
        }
        __syncwarp();

        // ---- part 3: bookkeeping, update, end of the pass ----
        bool upd = false;
        if (active) {
            if (search) {
                if (acc >= 0) miss = 0;
                else if (counted && ++miss > c.p.max_gap) end = true;
            }
            if (!end) {
                const uint16_t enew = acc >= 0 ? (uint16_t)(acc - dn.x) : kNoHit;
                if (UP || row < r0 || enew != eold) gt[row] = enew;
                upd = acc >= 0;
            }
        }
        __syncwarp();
        if (upd) {
            fit_update(f, ay, az, iwy, c);
            updates++;
            if (UP) { p0 = ay; p1 = az; p2 = f.s; p3 = f.t; p4 = f.q; top = row; }
            else { p0 = f.y; p1 = f.z; p2 = f.s; p3 = f.t; p4 = f.q; p5 = f.chi2; first = row; nh = f.n; }
        }
        __syncwarp();
        if (active && (end || row == (UP ? nr - 1 : 0))) {
            if (UP) {   // hand the tracklet to the down sweep: a fresh fit will start at its top hit
                UpRec r; r.y = p0; r.z = p1; r.s = p2; r.t = p3; r.q = p4; r.r0 = r0; r.top = top; r.id = i;
                float4* dst = reinterpret_cast<float4*>(&v.tl_up[i]);
                dst[0] = make_float4(r.y, r.z, r.s, r.t);
                dst[1] = make_float4(r.q, __int_as_float(r.r0), __int_as_float(r.top), __int_as_float(r.id));
                atomicAdd(&v.dn_count[tb + top], 1);
            } else {
                v.tl_rows[i] = first | (top << 8) | (nh << 16);
                const int sc = v.S_cap;
                v.tl_par[i] = p0; v.tl_par[sc + i] = p1; v.tl_par[2 * sc + i] = p2; v.tl_par[3 * sc + i] = p3;
                v.tl_par[4 * sc + i] = p4; v.tl_par[5 * sc + i] = p5;
            }
            ph = 0;
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&sm.empty[s]);
        it++;
    }
    unsigned long long vs = visits, us = updates;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { vs += __shfl_xor_sync(kFull, vs, o); us += __shfl_xor_sync(kFull, us, o); }
    if (lane == 0 && vs) { atomicAdd(&v.cnt[CNT_ROW_VISITS], vs); atomicAdd(&v.cnt[CNT_UPDATES], us); }
}

// parked tracklets -> lists by (task, top row) for the down sweep
__global__ void __launch_bounds__(256) k_dn_scatter(const View v, int nr) {
    const int S = min(v.seed_start[v.n_bins], v.S_cap);
    const int i = blockIdx.x * 256 + threadIdx.x;
    if (i >= S) return;
    const float4 a = reinterpret_cast<const float4*>(&v.tl_up[i])[0];
    const float4 b = reinterpret_cast<const float4*>(&v.tl_up[i])[1];
    const int r0 = __float_as_int(b.y), top = __float_as_int(b.z);
    const int bin = v.seed_bin[i] - r0 + top;
    const int pos = v.dn_start[bin] + atomicAdd(&v.dn_fill[bin], 1);
    float4* dst = reinterpret_cast<float4*>(&v.dn_rec[pos]);
    dst[0] = a; dst[1] = b;
}

}  // namespace tpc
