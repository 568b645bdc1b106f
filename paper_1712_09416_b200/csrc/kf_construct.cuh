// kf_construct.cuh -- K5 tracklet constructor: one CTA per sector task, pad rows in lock step, tracklet states in
// shared memory, row data staged by TMA bulk copies.
//
// A CTA takes a sector task and sweeps its pad rows twice: upwards for the up passes, then downwards for the down
// passes.  The rows -- hits and grid cell table of row r, one cp.async.bulk each, completion on an
// mbarrier -- go through a ring of kCtRing shared-memory slots, refilled by whichever warp is last through a row
// (there is no producer warp).  The Kalman state of every tracklet under way (32 words) lives in a shared-memory
// slot; at each row the CTA's 12 warps take the occupied slots 32 at a time, load the states, advance them by that row (transport, linked / recorded hit
// or window search in the staged row, update) and store them back.  All tracklets of the task are therefore at the
// same row at the same time, which is what the seed de-duplication needs (R23): an up pass marks every
// hit it records in a per-row bitmap; after a barrier the start hits of that row are taken in, and those already
// marked build no tracklet.  A tracklet whose up pass has ended is parked (its top hit and direction, 32 bytes);
// the down sweep takes the parked ones in kCtDnBatch rows at a time and starts each below its top row.  Nothing
// depends on which warp or slot a tracklet lands in.
//
// The arithmetic is that of kf_kernels.cuh (fit_transport / fit_update), so every decision is the one DESIGN.md
// "O5" describes.
#pragma once
#include "common.cuh"
#include "kf_kernels.cuh"

namespace tpc {

// 12 warps: 2 CTAs x 384 threads per SM leave 80 registers per thread (the register file is handed out per four
// warps of a CTA: a thirteenth warp would cost every warp 16 registers).  Measured on config 5 (K5 alone), with a
// producer warp: 13 + 1 warps (72 registers, 180 B of spills per thread, every spill an L2 round trip because the
// shared-memory carve-out leaves ~10 KB of L1) 5.82 ms; 9 + 1 warps at 96 registers 4.50 ms; without one: 8 warps
// 4.57 ms, 12 warps 4.40 ms.
#ifndef TPC_CT_WARPS
#define TPC_CT_WARPS 12
#endif
#ifndef TPC_CT_MINB
#define TPC_CT_MINB 2
#endif
#ifndef TPC_CT_RING
#define TPC_CT_RING 3
#endif
#ifndef TPC_CT_INL
#define TPC_CT_INL __forceinline__   // intake / turn inlined: 5.95 ms against 6.42 ms out of line (config 5)
#endif
constexpr int kCtWarps = TPC_CT_WARPS;                 // warps of a CTA, two CTAs per SM
constexpr int kCtWarpsWide = 20;                       // ... of the one-CTA-per-SM tiers (640 threads x 96 registers, no spills)
constexpr int ct_threads(int warps) { return warps * 32; }
constexpr int kCtRing = TPC_CT_RING;                   // rows in flight
#ifndef TPC_CT_DNB
#define TPC_CT_DNB 4
#endif
constexpr int kCtDnBatch = TPC_CT_DNB;                 // down sweep: the parked tracklets of this many rows are taken in at once
constexpr int kCtWords = 32;                           // 4-byte words of a tracklet's state
#ifndef TPC_CT_STAGE
#define TPC_CT_STAGE 48
#endif
constexpr int kCtSeedStage = TPC_CT_STAGE;             // start-hit records of a row staged with the row (more: read in place)
// State slots per sector task = tracklets under way at once, in three tiers (the host moves up one tier when a
// launch reports kErrSlotCapacity and stays there): shared-memory slots + slots in global memory (L2)
constexpr int kCtTiers = 3;
#ifndef TPC_CT_CAP0
#define TPC_CT_CAP0 512
#endif
#ifndef TPC_CT_SPILL0
#define TPC_CT_SPILL0 0
#endif
constexpr int kCtCapSmem[kCtTiers] = {TPC_CT_CAP0, 1408, 1280};   // tier 0: two CTAs per SM; tiers 1, 2: one
constexpr int kCtCapSpill[kCtTiers] = {TPC_CT_SPILL0, 0, 4096};
constexpr int kCtCapMax = 1280 + 4096;
#ifndef TPC_SW_CAP
#define TPC_SW_CAP 640
#endif
constexpr int kSwCap = TPC_SW_CAP;                            // hits of a row staged in shared memory; larger rows are read in place
constexpr int kSwHitBytes = (kSwCap + 2) * 8;          // + alignment slack of the bulk copy (16-byte granules)
constexpr int kSwCellEntries = kCellsPerHit * kSwCap + kCellPad + 16;
constexpr int kSwCellBytes = kSwCellEntries * 2;
static_assert(kSwHitBytes % 16 == 0 && kSwCellBytes % 16 == 0, "bulk copies are 16-byte granular");

// a start hit: its coordinates, the direction (sin phi, tg lambda) of the line to its up-link (DESIGN.md "O5" up pass,
// initial state), the hit itself, its up-link, and that one's
struct __align__(16) SeedRec { float y0, z0, s, t; int32_t h0, h1, h2, pad; };
// what the up pass hands down: its top hit, (sin phi, tg lambda, q/pT) there, start row | top row << 8, the table
// entry of the row below the top hit, the tracklet
struct __align__(16) UpRec { float y, z, s, t, q; int32_t rows, below, id; };

#ifndef TPC_CT_ROWS
#define TPC_CT_ROWS (TPC_MAX_ROWS + 1)
#endif
constexpr int kCtRows = TPC_CT_ROWS;
struct __align__(128) CtSmem {
    BinDesc desc[kCtRows];                    // the task's row descriptors
    unsigned char hits[kCtRing][kSwHitBytes];
    unsigned char cells[kCtRing][kSwCellBytes];
    SeedRec seeds[kCtRing][kCtSeedStage > 0 ? kCtSeedStage : 1];              // the first records of what starts at the row: start hits (up
                                                       // sweep), parked tracklets with their top hit there (down sweep)
    int32_t lo[kCtRows];                      // up sweep: first start hit of each row in the canonical list;
    int32_t cnt[kCtRows];                     // start hits of the row.  Down sweep: the same for the parked tracklets
    int32_t dcnt[kCtRows];                    // tracklets parked with their top hit in each row
    uint32_t used[2][TPC_MAX_ROW_HITS / 32];           // hits of the row at hand recorded by an up pass (double buffered)
    uint32_t occ[(kCtCapMax + 31) / 32];               // occupied state slots
    unsigned long long full[kCtRing], tbar;
    int32_t rel[kCtRing];                              // warps through with the row in the ring slot
    int32_t S, task, first, abort, n_free, n_hw, n_parked, top_max, i0;   // first: lowest row with a start hit; n_hw: highest slot used so far + 1
    uint32_t n_visits[20], n_updates[20], n_built, n_done;   // this CTA's share of the run's counters (per consumer warp)
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
// try_wait that lets the hardware suspend the warp for up to `ns` before it answers
__device__ __forceinline__ bool mbar_try_wait_hint(unsigned long long* b, uint32_t parity, uint32_t ns) {
    uint32_t ok;
    asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n selp.u32 %0, 1, 0, p;\n}"
                 : "=r"(ok) : "r"(smem_u32(b)), "r"(parity), "r"(ns) : "memory");
    return ok != 0;
}
// bounded wait: a lost signal ends the kernel with kErrHang instead of hanging the device.  Every warp of the CTA waits
// for the same signals in the same order (one per row step, the barriers of a row step come after its wait), so a
// signal that never comes is missed by ALL warps at the same step: the first to run out of patience raises the flag,
// the others see it within 64 polls, and all leave the sweep loop together -- none is left behind at a ct_bar.
__device__ __forceinline__ bool mbar_wait(unsigned long long* b, uint32_t parity, volatile int32_t* abort) {
    if (mbar_try_wait(b, parity)) return true;
    for (unsigned n = 0; n < (1u << 17); n++) {   // a waiting warp issues nothing until the phase completes or the hint runs out
        if (mbar_try_wait_hint(b, parity, 20000u)) return true;
        if ((n & 63u) == 63u && *abort) return false;
    }
    *abort = 1;
    return false;
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, unsigned long long* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
// barrier of the CTA's W warps
template <int W> __device__ __forceinline__ void ct_bar() { asm volatile("bar.sync 1, %0;" ::"n"(W * 32) : "memory"); }

__device__ __forceinline__ size_t cell_index(int base, int bin) { return (size_t)kCellsPerHit * base + (size_t)bin * kCellPad; }

// ---------------------------------------------------------------------------------------------------------
// The rows of a sweep go through the ring without a producer warp: the warp that is LAST to be through with a row
// refills the ring slot it has just freed with the row kCtRing steps ahead (one lane, three bulk copies).
// ---------------------------------------------------------------------------------------------------------
// Down sweep: the parked tracklets are taken in -- at a barrier of the warps -- not row by row but kCtDnBatch rows at a
// time, at the sweep's first row and at every row r with r % kCtDnBatch == kCtDnBatch - 1, for the rows
// r - r % kCtDnBatch .. r (their records are contiguous in dn_rec); a tracklet taken in early waits in its slot until
// the sweep has passed its top row.  Between two such rows the warps run on their own, up to a ring's depth apart.
__device__ __forceinline__ bool ct_dn_intake_row(const CtSmem& sm, int row, int& rlo, int& n) {
    if (row % kCtDnBatch != kCtDnBatch - 1 && row != *(volatile const int32_t*)&sm.top_max) return false;
    rlo = row - row % kCtDnBatch;
    n = sm.lo[row] + sm.cnt[row] - sm.lo[rlo];
    return n > 0;
}
// one lane: the row (hits, grid cell table, the records of what starts there) into the ring slot of iteration j
__device__ __forceinline__ void ct_issue(const View& v, CtSmem& sm, int row, bool down, int tb, uint32_t j) {
    const int s = (int)(j % kCtRing), S = sm.S;
    const BinDesc& d = sm.desc[row];
    const bool rowdata = d.n > 0 && d.n <= kSwCap;
    // records to stage: start hits of the row (not beyond the pool), or tracklets parked there
    int rlo = row, nd = 0;
    if (down) ct_dn_intake_row(sm, row, rlo, nd);
    const int ns = down ? min(nd, kCtSeedStage) : max(0, min(min(sm.cnt[row], kCtSeedStage), S - sm.lo[row]));
    const void* const recs = down ? (const void*)(v.dn_rec + sm.i0 + sm.lo[rlo]) : (const void*)(v.seed_rec + sm.lo[row]);
    if (rowdata || ns > 0) {
        const int offh = d.base & 1;
        const uint32_t hb = rowdata ? (uint32_t)((offh + d.n + 1) & ~1) * 8u : 0u;
        const size_t g = cell_index(d.base, tb + row);
        const int offc = (int)(g & 7);
        const uint32_t cb = rowdata ? (((uint32_t)(offc + d.ny * d.nz + 1) * 2u + 15u) & ~15u) : 0u;
        mbar_arrive_expect_tx(&sm.full[s], hb + cb + 32u * (uint32_t)ns);
        if (rowdata) {
            bulk_g2s(sm.hits[s], v.shit + (d.base - offh), hb, &sm.full[s]);
            bulk_g2s(sm.cells[s], v.cells + (g - offc), cb, &sm.full[s]);
        }
        if (ns > 0) bulk_g2s(sm.seeds[s], recs, 32u * (uint32_t)ns, &sm.full[s]);
    } else {
        mbar_arrive(&sm.full[s]);
    }
}

// warp 0, the other warps waiting at a barrier: all state slots free (the stack of free slots, lowest on top.
// Measured: preferring the slots of the warps' first groups is SLOWER -- a step takes as long as its slowest lane,
// and fuller groups have slower slowest lanes)
__device__ __forceinline__ void ct_reset_slots(CtSmem& sm, uint16_t* freel, int cap) {
    const int lane = lane_id();
    for (int k = lane; k < cap; k += 32) freel[k] = (uint16_t)(cap - 1 - k);
    for (int k = lane; k < (kCtCapMax + 31) / 32; k += 32) sm.occ[k] = 0u;
    if (lane == 0) { sm.n_free = cap; sm.n_hw = 0; }
}

// warp 0, the other warps waiting at a barrier: the next sector task and its tables (sm.task >= n_tasks: none left)
__device__ __forceinline__ void ct_next_task(const View& v, const Const& c, CtSmem& sm, uint16_t* freel, int cap, uint32_t& tphase) {
    const int lane = lane_id();
    const int nr = c.n_rows;
    int task = 0;
    if (lane == 0) task = (int)atomicAdd(&v.kf_cursor[0], 1ull);
    task = __shfl_sync(kFull, task, 0);
    if (task >= v.n_tasks) { if (lane == 0) sm.task = task; return; }
    const int tb = task * nr;
    if (lane == 0) {
        mbar_arrive_expect_tx(&sm.tbar, (uint32_t)nr * 32u);
        bulk_g2s(sm.desc, v.desc + tb, (uint32_t)nr * 32u, &sm.tbar);
        sm.task = task; sm.n_parked = 0; sm.top_max = -1; sm.i0 = v.seed_start[tb];
    }
    int f = nr;
    for (int r = lane; r < nr; r += 32) {
        const int lo = v.seed_start[tb + r], n = v.seed_start[tb + r + 1] - lo;
        sm.lo[r] = lo; sm.cnt[r] = n;
        if (n > 0) f = min(f, r);
    }
    for (int k = lane; k < 2 * (TPC_MAX_ROW_HITS / 32); k += 32) (&sm.used[0][0])[k] = 0u;
    for (int r = lane; r < kCtRows; r += 32) sm.dcnt[r] = 0;
    ct_reset_slots(sm, freel, cap);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) f = min(f, __shfl_xor_sync(kFull, f, o));
    if (lane == 0) {
        sm.first = f;
        if (!mbar_wait(&sm.tbar, tphase, &sm.abort)) sm.first = nr;   // (the flag is up: every warp leaves behind the next barrier)
    }
    tphase ^= 1u;
    __syncwarp();
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

// ---- a tracklet's state in its shared-memory slot: word k of slot s sits at st[k * cap + s] ----
struct CtTrk {
    Fit f;
    float p5;                       // up: two table entries (see the row step).  The state right after the last accepted
                                    // update (words 22..27 of the slot) is written there at an update and read at the end
                                    // of the pass only: it never sits in registers across the Kalman arithmetic
    int i;                          // tracklet = canonical start-hit number (batch-global)
    int cur;                        // up: the linked hit to come; down: table entry of the row below (read one row ahead)
    int nxt;                        // up: the hit linked above cur (read one link ahead)
    int ph, miss, r0, top, aux;     // ph 1 up/follow, 2 up/extend, 3 down; aux: up = row of cur, down = first row
};
// A slot's 32 words sit in eight groups of four: word k of slot s of a pool of `cap` slots is float
// ((k / 4) * cap + s) * 4 + k % 4, so that the 32 lanes of a warp move four words each with one conflict-free 16-byte
// access.  Groups: (y z s t) (q c00 c10 c11) (c20 c21 c22 c30) (c31 c32 c33 c40) (c41 c42 c43 c44)
// (chi2 n | snapshot y z) (snapshot s t q | p5) (i cur packed nxt).
__device__ __forceinline__ float* ct_word(float* B, int slot, int cap, int k) { return B + ((((k >> 2) * cap) + slot) << 2) + (k & 3); }
__device__ __forceinline__ void ct_load(CtTrk& t, float* B, int slot, int cap) {
    Fit& f = t.f;
    const float4 g0 = *reinterpret_cast<const float4*>(ct_word(B, slot, cap, 0));
    const float4 g1 = *reinterpret_cast<const float4*>(ct_word(B, slot, cap, 4));
    const float4 g2 = *reinterpret_cast<const float4*>(ct_word(B, slot, cap, 8));
    const float4 g3 = *reinterpret_cast<const float4*>(ct_word(B, slot, cap, 12));
    const float4 g4 = *reinterpret_cast<const float4*>(ct_word(B, slot, cap, 16));
    const float2 g5 = *reinterpret_cast<const float2*>(ct_word(B, slot, cap, 20));
    const float4 g7 = *reinterpret_cast<const float4*>(ct_word(B, slot, cap, 28));
    f.y = g0.x; f.z = g0.y; f.s = g0.z; f.t = g0.w;
    f.q = g1.x; f.c00 = g1.y; f.c10 = g1.z; f.c11 = g1.w;
    f.c20 = g2.x; f.c21 = g2.y; f.c22 = g2.z; f.c30 = g2.w;
    f.c31 = g3.x; f.c32 = g3.y; f.c33 = g3.z; f.c40 = g3.w;
    f.c41 = g4.x; f.c42 = g4.y; f.c43 = g4.z; f.c44 = g4.w;
    f.chi2 = g5.x; f.n = __float_as_int(g5.y);
    t.p5 = *ct_word(B, slot, cap, 27);
    t.i = __float_as_int(g7.x); t.cur = __float_as_int(g7.y); t.nxt = __float_as_int(g7.w);
    const uint32_t pk = __float_as_uint(g7.z);
    t.ph = pk & 3u; t.miss = (pk >> 2) & 63u; t.r0 = (pk >> 8) & 255u; t.top = (pk >> 16) & 255u; t.aux = pk >> 24;
}
// first: the slot is being filled (word 28, the tracklet, never changes afterwards)
__device__ __forceinline__ void ct_store(const CtTrk& t, float* B, int slot, int cap, bool up, bool first = false) {
    const Fit& f = t.f;
    *reinterpret_cast<float4*>(ct_word(B, slot, cap, 0)) = make_float4(f.y, f.z, f.s, f.t);
    *reinterpret_cast<float4*>(ct_word(B, slot, cap, 4)) = make_float4(f.q, f.c00, f.c10, f.c11);
    *reinterpret_cast<float4*>(ct_word(B, slot, cap, 8)) = make_float4(f.c20, f.c21, f.c22, f.c30);
    *reinterpret_cast<float4*>(ct_word(B, slot, cap, 12)) = make_float4(f.c31, f.c32, f.c33, f.c40);
    *reinterpret_cast<float4*>(ct_word(B, slot, cap, 16)) = make_float4(f.c41, f.c42, f.c43, f.c44);
    *reinterpret_cast<float2*>(ct_word(B, slot, cap, 20)) = make_float2(f.chi2, __int_as_float(f.n));
    *ct_word(B, slot, cap, 27) = t.p5;
    if (first) *ct_word(B, slot, cap, 28) = __int_as_float(t.i);
    if (up) *ct_word(B, slot, cap, 29) = __int_as_float(t.cur);   // down: written by the asynchronous copy of the table word (see the row step)
    // word 31 (nxt): written at the intake and by the asynchronous copy of the next link
    *ct_word(B, slot, cap, 30) = __uint_as_float((uint32_t)t.ph | ((uint32_t)t.miss << 2) | ((uint32_t)t.r0 << 8) |
                                                 ((uint32_t)t.top << 16) | ((uint32_t)t.aux << 24));
}

// slot -> where its state lives: the first cap_s slots in shared memory, the others in this CTA's stretch of
// global memory (both multiples of 32, so a warp's 32 slots are all of one kind)
template <bool G, int CAPS>   // G: the tier has slots in global memory; CAPS: its slots in shared memory (a compile-time
struct CtSlots {              // constant: the words of a slot are then at fixed offsets from one address)
    static constexpr int cap_s = CAPS;
    float* st; float* gs; int cap_g;
    __device__ __forceinline__ void load(CtTrk& t, int slot) const {
        if (!G || slot < cap_s) ct_load(t, st, slot, cap_s); else ct_load(t, gs, slot - cap_s, cap_g);
    }
    __device__ __forceinline__ void store(const CtTrk& t, int slot, bool up, bool first = false) const {
        if (!G || slot < cap_s) ct_store(t, st, slot, cap_s, up, first); else ct_store(t, gs, slot - cap_s, cap_g, up, first);
    }
    // word k of a slot
    __device__ __forceinline__ float* word(int slot, int k) const {
        if (!G || slot < cap_s) return ct_word(st, slot, cap_s, k);
        return ct_word(gs, slot - cap_s, cap_g, k);
    }
    // word k of a slot := the 4 bytes at src, without waiting for them: an asynchronous copy for a slot in shared memory
    // (the warp waits for its copies when it is through with the row), a plain load and store for one in global memory
    __device__ __forceinline__ void fetch(int slot, int k, const void* src) const {
        if (!G || slot < cap_s) {
            asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_u32(ct_word(st, slot, cap_s, k))), "l"(src) : "memory");
        } else {
            *ct_word(gs, slot - cap_s, cap_g, k) = __ldg(reinterpret_cast<const float*>(src));
        }
    }
    // the state right after the last accepted update: words 22, 23 (y, z) and 24..27 (sin phi, tg lambda, q/pT, p5)
    __device__ __forceinline__ void snap_put(int slot, float y, float z, float s, float t, float q, float p5) const {
        *reinterpret_cast<float2*>(word(slot, 22)) = make_float2(y, z);
        *reinterpret_cast<float4*>(word(slot, 24)) = make_float4(s, t, q, p5);
    }
    __device__ __forceinline__ void snap_get(int slot, float& y, float& z, float& s, float& t, float& q) const {
        const float2 a = *reinterpret_cast<const float2*>(word(slot, 22));
        const float4 b = *reinterpret_cast<const float4*>(word(slot, 24));
        y = a.x; z = a.y; s = b.x; t = b.y; q = b.z;
    }
};

// take a state slot for every lane that asks; -1 when the task has more tracklets under way than slots
__device__ __forceinline__ int ct_pop(const View& v, CtSmem& sm, const uint16_t* freel, bool need, int cap) {
    const unsigned m = __ballot_sync(kFull, need);
    if (!m) return -1;
    int old = 0;
    if (lane_id() == 0) old = atomicSub(&sm.n_free, __popc(m));
    old = __shfl_sync(kFull, old, 0);
    if (!need) return -1;
    const int idx = old - 1 - __popc(m & lanemask_lt());
    if (idx < 0 || idx >= cap) { atomicOr((unsigned int*)&v.cnt[CNT_ERR], kErrSlotCapacity); return -1; }
    const int slot = freel[idx];
    atomicOr(&sm.occ[slot >> 5], 1u << (slot & 31));
    atomicMax(&sm.n_hw, slot + 1);
    return slot;
}
__device__ __forceinline__ void ct_push(CtSmem& sm, uint16_t* freel, int slot, int cap) {
    const int idx = atomicAdd(&sm.n_free, 1);
    if (idx >= 0 && idx < cap) freel[idx] = (uint16_t)slot;
}

// ---- intake, by all consumer threads between the row steps ----
// down sweep: the parked tracklets whose top hit is in this row start a fresh fit there (their records come
// ordered by top row: staged in the ring slot, the ones beyond kCtSeedStage read in place)
template <int W, bool G, int CAPS>
__device__ TPC_CT_INL void ct_intake_down(const View& v, const Const& c, CtSmem& sm, const CtSlots<G, CAPS>& sl, const uint16_t* freel,
                                            int cap, int rlo, int n, int s) {
    const int lo = sm.i0 + sm.lo[rlo];
    for (int j0 = 0; j0 < n; j0 += W * 32) {
        const int j = j0 + (int)threadIdx.x;
        const int slot = ct_pop(v, sm, freel, j < n, cap);
        if (slot >= 0) {
            float4 a4, b4;
            if (j < kCtSeedStage) {
                a4 = *reinterpret_cast<const float4*>(&sm.seeds[s][j]);
                b4 = *(reinterpret_cast<const float4*>(&sm.seeds[s][j]) + 1);
            } else {
                a4 = __ldcg(reinterpret_cast<const float4*>(&v.dn_rec[lo + j]));
                b4 = __ldcg(reinterpret_cast<const float4*>(&v.dn_rec[lo + j]) + 1);
            }
            CtTrk t;
            t.p5 = 0.f;
            const int top = (__float_as_int(b4.y) >> 8) & 0xff;
            t.r0 = __float_as_int(b4.y) & 0xff; t.top = top; t.i = __float_as_int(b4.w);
            t.f.y = a4.x; t.f.z = a4.y; t.f.s = a4.z; t.f.t = a4.w; t.f.q = b4.x;
            fit_prior(t.f, c); t.f.n = 1;
            t.aux = top; t.miss = 0; t.ph = 3; t.nxt = -1;
            t.cur = 0;
            sl.store(t, slot, false, true);
            {   // table entry of the row below the top hit, in both halves of the word (see the row step)
                const uint32_t below = (uint32_t)__float_as_int(b4.z) & 0xffffu;
                *sl.word(slot, 29) = __uint_as_float(below | (below << 16));
            }
            sl.snap_put(slot, a4.x, a4.y, a4.z, a4.w, b4.x, t.p5);
        }
    }
}
// up sweep: the start hits of this row that no up pass has recorded build a tracklet; returns how many (this thread)
template <int W, bool G, int CAPS>
__device__ TPC_CT_INL void ct_intake_up(const View& v, const Const& c, CtSmem& sm, const CtSlots<G, CAPS>& sl, const uint16_t* freel,
                                              int cap, int row, int s, int S) {
    const int D = c.p.link_step;
    const bool dedup = c.p.seed_dedup != 0;
    const int n = sm.cnt[row], lo = sm.lo[row], base = sm.desc[row].base;
    const uint32_t* const ub = sm.used[row & 1];
    for (int j0 = 0; j0 < n; j0 += W * 32) {
        const int j = j0 + (int)threadIdx.x, e = lo + j;
        bool need = false;
        int hl = 0;
        float4 a4 = make_float4(0.f, 0.f, 0.f, 0.f);
        int4 hh = make_int4(0, 0, 0, 0);
        if (j < n && e < S) {
            if (j < kCtSeedStage) {
                a4 = *reinterpret_cast<const float4*>(&sm.seeds[s][j]);
                hh = *(reinterpret_cast<const int4*>(&sm.seeds[s][j]) + 1);
            } else {
                a4 = __ldg(reinterpret_cast<const float4*>(&v.seed_rec[e]));
                hh = __ldg(reinterpret_cast<const int4*>(&v.seed_rec[e]) + 1);
            }
            hl = hh.x - base;
            if (dedup && ((ub[hl >> 5] >> (hl & 31)) & 1u)) v.tl_rows[e] = 0;   // skipped: n_hits = 0
            else need = true;
        }
        const int slot = ct_pop(v, sm, freel, need, cap);
        if (need && slot < 0) v.tl_rows[e] = 0;
        if (slot >= 0) {
            atomicAdd(&sm.n_built, 1u);
            CtTrk t;
            Fit& f = t.f;
            f.y = a4.x; f.z = a4.y; f.s = a4.z; f.t = a4.w; f.q = 0.f;   // direction of the first link, from K4
            fit_prior(f, c); f.n = 0;
            t.p5 = __uint_as_float(((uint32_t)kNoHit << 16) | (uint32_t)hl);   // table entries: below the top hit | of the row before
            t.i = e; t.cur = hh.y; t.nxt = hh.z; t.ph = 1; t.miss = 0; t.r0 = row; t.top = row; t.aux = row + D;
            v.tl_tab[(size_t)e * v.tab_stride + row] = (uint16_t)hl;
            sl.store(t, slot, true, true);
            *sl.word(slot, 31) = __int_as_float(t.nxt);
            sl.snap_put(slot, a4.x, a4.y, a4.z, a4.w, 0.f, t.p5);
        }
    }
}
// between the sweeps (all warps): the parked tracklets of the task, ordered by top row, into dn_rec
template <int W>
__device__ TPC_CT_INL void ct_turn(const View& v, CtSmem& sm, int nr) {
    const int lane = lane_id(), warp = threadIdx.x >> 5;
    if (warp == 0) {   // lo = exclusive scan of the counts, cnt = the counts, dcnt = 0 (fill counters of the scatter)
        int carry = 0;
        for (int r0 = 0; r0 < nr; r0 += 32) {
            const int r = r0 + lane;
            const int c = r < nr ? sm.dcnt[r] : 0;
            int incl = c;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { const int x = __shfl_up_sync(kFull, incl, o); if (lane >= o) incl += x; }
            if (r < nr) { sm.lo[r] = carry + incl - c; sm.cnt[r] = c; sm.dcnt[r] = 0; }
            carry += __shfl_sync(kFull, incl, 31);
        }
    }
    ct_bar<W>();
    const uint32_t* const plist = v.kf_park + sm.i0;
    const int np = sm.n_parked;
    for (int k = threadIdx.x; k < np; k += W * 32) {
        const uint32_t w = __ldcg(&plist[k]);
        const int top = (int)(w >> 24), id = sm.i0 + (int)(w & 0xffffffu);
        const int pos = sm.lo[top] + atomicAdd(&sm.dcnt[top], 1);
        const float4 a4 = __ldcg(reinterpret_cast<const float4*>(&v.tl_up[id]));
        const float4 b4 = __ldcg(reinterpret_cast<const float4*>(&v.tl_up[id]) + 1);
        float4* dst = reinterpret_cast<float4*>(&v.dn_rec[sm.i0 + pos]);
        dst[0] = a4; dst[1] = b4;
    }
    asm volatile("fence.proxy.async;" ::: "memory");   // the bulk copies (async proxy) will read these records
    ct_bar<W>();
}

// ---------------------------------------------------------------------------------------------------------
// K5
// ---------------------------------------------------------------------------------------------------------
template <int W, bool G, int CAPS>
#ifdef TPC_CT_MAXNREG
__global__ void __maxnreg__(TPC_CT_MAXNREG) k_construct(
#else
__global__ void __launch_bounds__(W * 32, W <= 16 ? TPC_CT_MINB : 1) k_construct(
#endif
const __grid_constant__ View v, const __grid_constant__ Const c, const int cap_g, float* const spill) {
    constexpr int cap_s = CAPS;
    extern __shared__ __align__(128) unsigned char ct_raw[];
    TPC_RETURN_IF_REJECTED(v);
    CtSmem& sm = *reinterpret_cast<CtSmem*>(ct_raw);
    const int cap = cap_s + cap_g;
    CtSlots<G, CAPS> sl;
    sl.st = reinterpret_cast<float*>(ct_raw + sizeof(CtSmem)); sl.cap_g = cap_g;
    sl.gs = spill + (size_t)blockIdx.x * kCtWords * cap_g;
    uint16_t* const freel = reinterpret_cast<uint16_t*>(sl.st + (size_t)kCtWords * cap_s);   // stack of free slots
    const int warp = threadIdx.x >> 5, lane = lane_id();
    if (threadIdx.x == 0) {
        for (int s = 0; s < kCtRing; s++) { mbar_init(&sm.full[s], 1); sm.rel[s] = 0; }
        mbar_init(&sm.tbar, 1);
        sm.abort = 0; sm.n_built = 0u; sm.n_done = 0u; sm.S = min(v.seed_start[v.n_bins], v.S_cap);   // start hits of the batch
        for (int k = 0; k < 20; k++) { sm.n_visits[k] = 0u; sm.n_updates[k] = 0u; }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const int nr = c.n_rows, D = c.p.link_step;
    volatile int32_t* const abort = &sm.abort;
    uint32_t it = 0, tphase = 0;      // rows through the ring so far (the same count in every warp); phase of tbar (warp 0)
    int phase = 0;                    // 0: a sector task is due; 1: up sweep; 2: down sweep
    int row = 0, last = 0, tb = 0;    // the row at hand, the last row of the sweep, the task's first bin

    for (;;) {
        if (phase == 0) {
            ct_bar<W>();                                         // every warp is through with the task before
            if (warp == 0) ct_next_task(v, c, sm, freel, cap, tphase);
            ct_bar<W>();
            const int task = *(volatile int32_t*)&sm.task;
            if (task >= v.n_tasks || *abort) break;               // (the flag is read behind a barrier: the same in every warp)
            tb = task * nr;
            row = *(volatile int32_t*)&sm.first; last = nr - 1;
            if (row > last) continue;                            // no start hit in this sector
            phase = 1;
            if (warp == 0 && lane == 0)                          // the ring is empty: its first rows
                for (int k = 0; k < kCtRing; k++) if (row + k <= last) ct_issue(v, sm, row + k, false, tb, it + k);
        }
        const bool up = phase == 1;
        const int s = (int)(it % kCtRing);
        if (!mbar_wait(&sm.full[s], (it / kCtRing) & 1u, abort)) break;
        const BinDesc& dsc = sm.desc[row];
        const int4 dn = make_int4(dsc.base, dsc.n, dsc.ny, dsc.nz);
        const bool staged = dn.y <= kSwCap;
        const size_t cg = cell_index(dn.x, tb + row);
        const float2* const hits = staged ? reinterpret_cast<const float2*>(sm.hits[s]) + (dn.x & 1) : v.shit + dn.x;
        const uint16_t* const cs = staged ? reinterpret_cast<const uint16_t*>(sm.cells[s]) + (cg & 7) : v.cells + cg;

        // The warps meet at barriers only around an intake: rows where nothing starts (most rows of a sparse
        // event) are processed by every warp on its own, up to a ring's depth apart.
        const bool intake = sm.cnt[row] > 0;
        int dn_lo = 0, dn_n = 0;
        if (!up && ct_dn_intake_row(sm, row, dn_lo, dn_n)) {   // down sweep: what starts at these rows is taken in BEFORE
            ct_bar<W>();                                        // this row is processed; all slots freed by the rows above
            ct_intake_down<W, G, CAPS>(v, c, sm, sl, freel, cap, dn_lo, dn_n, s);   // are back on the stack
            ct_bar<W>();
        }
        // ---- one pad row for the tracklets under way: the warps share the groups of 32 slots ----
        const int n_groups = (*(volatile int32_t*)&sm.n_hw + 31) >> 5;
        for (int g = warp; g < n_groups; g += W) {
            const uint32_t occ = *(volatile uint32_t*)&sm.occ[g];
            if (!occ) continue;
            const int slot = (g << 5) + lane;
            bool on = (occ >> lane) & 1u;
            CtTrk t;
            if (on) sl.load(t, slot);
            if (on && !up && t.top <= row) on = false;          // starts below its top row
            Fit& f = t.f;
            uint16_t* const gt = v.tl_tab + (size_t)(on ? t.i : 0) * v.tab_stride;
            bool end = false, search = false, counted = false, vis = false;
            int acc = -1;
            uint16_t eold = kNoHit;
            float ay = 0.f, az = 0.f, iwy = 0.f, iwz = 0.f;
            // part 1: transport and the candidate that is already known
            if (on) {
                int known = -1;
                float ky = 0.f, kz = 0.f;
                if (up) {
                    if (t.ph == 1 && row == t.aux) {
                        known = t.cur;
                        const float2 hk = hits[t.cur - dn.x]; ky = hk.x; kz = hk.y;
                    }
                } else if (row >= t.r0) {
                    // the slot's word 29 holds the 4-byte word of the tracklet's table with this row's entry; the one with
                    // the entry of the row below is fetched now and read at the next row
                    eold = (uint16_t)((uint32_t)t.cur >> (16 * (row & 1)));
                    if (row > t.r0) sl.fetch(slot, 29, gt + ((row - 1) & ~1));
                    if (eold != kNoHit) { known = dn.x + eold; const float2 hk = hits[eold]; ky = hk.x; kz = hk.y; }
                }
                end = !fit_transport(f, c.row_x[up ? row - 1 : row + 1], c.row_x[row], c);
                if (!end) {
                    vis = true;
                    iwy = 1.f / (f.c00 + c.sigma_y2); iwz = 1.f / (f.c11 + c.sigma_z2);
                    bool gate_ok = false;
                    if (known >= 0) {   // the gate value of (ky, kz) on the predicted state
                        const float ry = ky - f.y, rz = kz - f.z;
                        gate_ok = (ry * ry) * iwy + (rz * rz) * iwz <= c.p.chi2_link;
                        if (gate_ok) { acc = known; ay = ky; az = kz; }
                    }
                    if (up) {
                        if (t.ph == 1) {
                            if (row == t.aux) {
                                // the link above the next linked hit (needed one link from now) is fetched into the slot
                                if (gate_ok && t.nxt >= 0) sl.fetch(slot, 31, &v.clink_up[t.nxt]);
                                if (gate_ok) { t.cur = t.nxt; t.aux += D; if (t.cur < 0) t.ph = 2; }
                                else { t.ph = 2; search = true; counted = true; }
                            }   // else: in-between row of a step-2 link
                        } else {
                            search = true; counted = true;
                        }
                    } else {
                        search = row < t.r0 || known < 0;
                        counted = row < t.r0;
                    }
                    if (search && counted && fabsf(f.y) > c.row_x[row] * c.tan_half_angle + c.p.edge_margin) {
                        end = true; search = false;
                    }
                }
            }
            // part 2: the window searches of this row
            __syncwarp();
            if (search && dn.y > 0) {
                const float4 gf = make_float4(dsc.y0, dsc.z0, dsc.idy, dsc.idz);
                float bg = 0.f;   // a lane that searches has accepted nothing yet on this row: (ay, az) are free
                const int bp = sweep_search(v, c, f, gf, dn, hits, cs, iwy, iwz, ay, az, bg);
                if (bp >= 0 && bg <= c.p.chi2_ext) acc = dn.x + bp;
            }
            __syncwarp();
            // part 3: bookkeeping, update, end of the pass
            bool upd = false;
            if (on) {
                if (search) {
                    if (acc >= 0) t.miss = 0;
                    else if (counted && ++t.miss > c.p.max_gap) end = true;
                }
                if (!end) {
                    const uint16_t enew = acc >= 0 ? (uint16_t)(acc - dn.x) : kNoHit;
                    if (up || row < t.r0 || enew != eold) gt[row] = enew;
                    upd = acc >= 0;
                    if (up) {   // p5 = table entry below the top hit << 16 | entry of the row before this one -> of this one
                        const uint32_t q = __float_as_uint(t.p5);
                        t.p5 = __uint_as_float((upd ? q << 16 : q & 0xffff0000u) | enew);
                    }
                }
            }
            __syncwarp();
            if (upd) {
                fit_update(f, ay, az, iwy, c);
                if (up) {
                    sl.snap_put(slot, ay, az, f.s, f.t, f.q, t.p5); t.top = row;
                    if (intake) {                               // seed de-duplication: this hit is being followed
                        const int hl = acc - dn.x;              // (marks matter only where start hits wait)
                        atomicOr(&sm.used[row & 1][hl >> 5], 1u << (hl & 31));
                    }
                } else {
                    t.p5 = f.chi2; t.aux = row;
                    sl.snap_put(slot, f.y, f.z, f.s, f.t, f.q, t.p5);
                }
            }
            __syncwarp();
            const bool fin = on && (end || row == (up ? nr - 1 : 0));
            if (fin) {
                float p0, p1, p2, p3, p4;
                sl.snap_get(slot, p0, p1, p2, p3, p4);
                if (up) {   // park: a fresh fit will start at the top hit in the down sweep
                    float4* dst = reinterpret_cast<float4*>(&v.tl_up[t.i]);
                    const int below = t.top > t.r0 ? (int)(__float_as_uint(t.p5) >> 16) : (int)kNoHit;
                    dst[0] = make_float4(p0, p1, p2, p3);
                    dst[1] = make_float4(p4, __int_as_float(t.r0 | (t.top << 8)), __int_as_float(below), __int_as_float(t.i));
                    const int k = atomicAdd(&sm.n_parked, 1);
                    v.kf_park[sm.i0 + k] = (uint32_t)(t.i - sm.i0) | ((uint32_t)t.top << 24);   // in order of parking
                    atomicAdd(&sm.dcnt[t.top], 1);
                    atomicMax(&sm.top_max, t.top);
                } else {
                    v.tl_rows[t.i] = t.aux | (t.top << 8) | (f.n << 16);
                    const int sc = v.S_cap;
                    v.tl_par[t.i] = p0; v.tl_par[sc + t.i] = p1; v.tl_par[2 * sc + t.i] = p2; v.tl_par[3 * sc + t.i] = p3;
                    v.tl_par[4 * sc + t.i] = p4; v.tl_par[5 * sc + t.i] = t.p5;
                }
            } else if (on) {
                sl.store(t, slot, up);
            }
            const unsigned gone = __ballot_sync(kFull, fin);    // this warp alone owns the group's occupancy word now
            const unsigned nvis = __popc(__ballot_sync(kFull, vis)), nupd = __popc(__ballot_sync(kFull, upd));
            if (lane == 0) {
                if (gone) sm.occ[g] = occ & ~gone;
                sm.n_visits[warp] += nvis; sm.n_updates[warp] += nupd;
            }
            if (fin) ct_push(sm, freel, slot, cap);
        }
        asm volatile("cp.async.wait_all;" ::: "memory");   // this warp's fetches into its slots have landed
        // up sweep: the start hits of this row are taken in AFTER it is processed (its marks are complete); the marks'
        // other buffer is cleared here for the next row if start hits wait there (its last readers, the intake two rows
        // down, are behind that row's barriers)
        const bool next_intake = up && row + 1 < nr && sm.cnt[row + 1] > 0;
        if (up && (intake || next_intake)) {
            ct_bar<W>();
            if (intake) ct_intake_up<W, G, CAPS>(v, c, sm, sl, freel, cap, row, s, sm.S);
            if (next_intake)
                for (int k = threadIdx.x; k < TPC_MAX_ROW_HITS / 32; k += W * 32) sm.used[(row + 1) & 1][k] = 0u;
            ct_bar<W>();
        }
        // through with the row: the last warp refills the ring slot with the row kCtRing steps ahead
        __syncwarp();
        if (lane == 0) {
            __threadfence_block();
            if (atomicAdd(&sm.rel[s], 1) == W - 1) {
                sm.rel[s] = 0;
                const int r2 = up ? row + kCtRing : row - kCtRing;
                if (up ? r2 <= last : r2 >= last) ct_issue(v, sm, r2, !up, tb, it + kCtRing);
            }
        }
        it++;
        if (row != last) { row += up ? 1 : -1; continue; }
        if (!up) { phase = 0; continue; }
        // the turn: every warp is through with the up sweep; the parked tracklets are ordered by top row (lo / cnt
        // become theirs), all slots are free again, and the down sweep starts from the highest top row
        ct_bar<W>();
        if (warp == 0) ct_reset_slots(sm, freel, cap);
        ct_turn<W>(v, sm, nr);
        row = *(volatile int32_t*)&sm.top_max; last = 0;
        if (row < 0) { phase = 0; continue; }
        phase = 2;
        if (warp == 0 && lane == 0)
            for (int k = 0; k < kCtRing; k++) if (row - k >= 0) ct_issue(v, sm, row - k, true, tb, it + k);
    }
    __syncwarp();
    if (lane == 0) {
        if (warp == 0 && *abort) atomicOr((unsigned int*)&v.cnt[CNT_ERR], kErrHang);   // the host reports it (TPC_ERR_CUDA)
        const uint32_t vs = sm.n_visits[warp], us = sm.n_updates[warp];
        if (vs) { atomicAdd(&v.cnt[CNT_ROW_VISITS], (unsigned long long)vs); atomicAdd(&v.cnt[CNT_UPDATES], (unsigned long long)us); }
        __threadfence_block();
        if (atomicAdd(&sm.n_done, 1u) == (uint32_t)(W - 1)) {   // the last consumer warp out
            const uint32_t bs = *(volatile uint32_t*)&sm.n_built;
            if (bs) atomicAdd(&v.cnt[CNT_TRACKLETS], (unsigned long long)bs);
        }
    }
}

// the three tiers
#define TPC_K5_TIER0 k_construct<kCtWarps, (kCtCapSpill[0] > 0), kCtCapSmem[0]>
#define TPC_K5_TIER1 k_construct<kCtWarpsWide, false, kCtCapSmem[1]>
#define TPC_K5_TIER2 k_construct<kCtWarpsWide, true, kCtCapSmem[2]>

}  // namespace tpc
