// tracker.cu -- host side of libtpctrack.so: the C ABI of include/tpctrack.h, work-space management and the
// launch sequence K1..K6 for a batch of events (all n_events * n_sectors sector tasks in every launch).
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include "ca_kernels.cuh"
#include "kf_kernels.cuh"
#include "kf_construct.cuh"
#include "sel_kernels.cuh"
#include "kf_refit.cuh"
#include "merge_kernels.cuh"
#include "kf_global.cuh"
#include "peak_kernels.cuh"

namespace {

// int32 / float arrays per track: 4 + next, prev, global + global fit (ndf, hits, sector); 7 + the outer state (6) + the
// global fit (7)
constexpr int kOutI = 10, kOutF = 20;
constexpr int kOutI_plain = 4, kOutF_plain = 7, kOutF_refit = 13;
constexpr int kAsync = 3;              // batches in flight through tpc_submit_events

thread_local std::string g_err;

void set_err(const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    g_err = buf;
}

#define CK(call)                                                                       \
    do {                                                                               \
        cudaError_t e_ = (call);                                                       \
        if (e_ != cudaSuccess) {                                                       \
            set_err("%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); \
            return TPC_ERR_CUDA;                                                       \
        }                                                                              \
    } while (0)

// a device (or pinned host) array that only ever grows
template <class T> struct Buf {
    T* p = nullptr;
    size_t cap = 0;
    bool host = false;
    int reserve(size_t n) {
        if (n <= cap) return TPC_OK;
        release();
        const size_t want = n + n / 8 + 64;
        cudaError_t e = host ? cudaMallocHost((void**)&p, want * sizeof(T)) : cudaMalloc((void**)&p, want * sizeof(T));
        if (e != cudaSuccess) {
            p = nullptr; cap = 0;
            set_err("allocation of %zu bytes failed: %s", want * sizeof(T), cudaGetErrorString(e));
            return TPC_ERR_CUDA;
        }
        cap = want;
        return TPC_OK;
    }
    void release() {
        if (p) { if (host) cudaFreeHost(p); else cudaFree(p); }
        p = nullptr; cap = 0;
    }
};

}  // namespace

using namespace tpc;

// Work space and state of one group of events in flight: every kernel launch covers all its sector tasks.
struct Batch {
    cudaStream_t stream = nullptr;           // the stream this group runs on
    View v;
    int n_events = 0, first_event = 0;
    int64_t N = 0, S_cap = 0;
    bool host_in = false;
    const tpc_event_in* in = nullptr;
    std::vector<int32_t> ev_n, ev_off;       // clusters per event, offset in the group
    tpc_counters counters;                   // of the group's last run
    // device pools
    Buf<float> in_x, in_y, in_z, tl_par, o_f[kOutF];
    Buf<float2> shit;
    Buf<float4> thit;
    Buf<int32_t> in_row, sec_off, bin_count, bin_start, tidx, sorig, link_up, link_dn, clink_up, clink_dn, seed_count,
        seed_start, seeds, seed_bin, tl_rows, tl_nown, tl_keep, trk_scan, hit_scan, ev_off_d,
        o_i[kOutI], o_hit, trk_rows, trk_task, mg_list;
    Buf<unsigned long long> mg_next, mg_prev, scratch;
    Buf<uint16_t> slot, cells, tl_tab;
    Buf<float2> o_hit_yz;
    Buf<uint8_t> o_hit_row;
    Buf<int32_t> trk_hit0;
    Buf<BinDesc> desc;
    Buf<SeedRec> seed_rec;
    Buf<UpRec> tl_up, dn_rec;
    Buf<uint32_t> kf_park;
    Buf<int32_t> dn_count, dn_start, dn_fill, tl_cnt;
    int sel_C = 1;                           // selector chunks per sector task
    int ct_tier = 0;                         // K5 slot tier used by this group's last launch
    Buf<float> ct_spill;                     // tier 2: state slots in global memory, per CTA of THIS group's launch (groups
                                             // and tickets run on streams of their own: their K5 launches can be resident together)
    // the launch sequence K1..K6 (+ refit, merge) of this group as a CUDA graph, replayed while nothing it bakes in changes
    // Two graphs are kept: with device inputs a ticket's output arrays alternate between two sets (tpc_wait_events swaps
    // them with the ticket's), so consecutive runs of one shape need two graphs, not a new capture each time.
    struct GraphKey { View v; int tier, maxn, n_events; int64_t S_cap; const float* spill; };
    static constexpr int kGraphs = 2;
    GraphKey gkey[kGraphs];
    cudaGraphExec_t gexec[kGraphs] = {};
    int64_t graph_launches[kGraphs] = {};    // kernels in each graph
    int graph_victim = 0;                    // the graph that a new shape replaces
    Buf<uint32_t> owner;
    Buf<EventSrc> ev_src;
    Buf<unsigned long long> cnt, kf_cursor;
    // pinned host mirrors
    Buf<EventSrc> h_ev_src;
    Buf<int32_t> h_sec_off, h_ev_off, h_nseeds;
    Buf<unsigned long long> h_cnt;
    cudaEvent_t evt[TPC_N_STAGES + 1] = {};
    cudaEvent_t kernels_done = nullptr;      // recorded behind the last kernel of a run (submit / wait pipeline)
    cudaEvent_t wait_for = nullptr;          // the kernels of this run start behind this event (another batch's kernels)
    float stage_ms[TPC_N_STAGES] = {};

    Batch() {
        h_ev_src.host = h_sec_off.host = h_ev_off.host = h_cnt.host = h_nseeds.host = true;
        memset(&v, 0, sizeof v);
        memset(&counters, 0, sizeof counters);
    }
    void free_all() {
        in_x.release(); in_y.release(); in_z.release(); thit.release(); shit.release(); tl_par.release();
        for (auto& b : o_f) b.release();
        in_row.release(); sec_off.release(); bin_count.release(); bin_start.release(); tidx.release(); sorig.release();
        link_up.release(); link_dn.release(); clink_up.release(); clink_dn.release(); seed_count.release();
        seed_start.release(); seeds.release(); seed_bin.release(); tl_tab.release(); tl_rows.release();
        tl_nown.release(); tl_keep.release(); trk_scan.release(); hit_scan.release(); ev_off_d.release();
        scratch.release(); o_hit.release();
        for (auto& b : o_i) b.release();
        slot.release(); cells.release(); desc.release(); owner.release(); ev_src.release();
        seed_rec.release(); tl_up.release(); dn_rec.release(); kf_park.release(); dn_count.release(); dn_start.release(); dn_fill.release(); tl_cnt.release(); o_hit_yz.release(); o_hit_row.release(); trk_hit0.release(); trk_rows.release(); trk_task.release(); mg_next.release(); mg_prev.release(); mg_list.release();
        cnt.release(); kf_cursor.release(); ct_spill.release(); h_ev_src.release(); h_sec_off.release(); h_ev_off.release(); h_cnt.release(); h_nseeds.release();
        for (auto& e : evt) if (e) { cudaEventDestroy(e); e = nullptr; }
        if (kernels_done) { cudaEventDestroy(kernels_done); kernels_done = nullptr; }
        for (auto& g : gexec) if (g) { cudaGraphExecDestroy(g); g = nullptr; }
    }
};

struct tpc_tracker {
    Const c;
    std::vector<float> sector_alpha;
    cudaStream_t user_stream = nullptr;      // tpc_tracker_set_stream: used by slot 0 when the call is one group
    std::vector<cudaStream_t> own_streams;   // one per slot
    int sm_count = 148;
    int ct_tier = 0;                         // K5: state-slot tier (kf_construct.cuh); moves up on kErrSlotCapacity
    int ct_blocks[kCtTiers] = {296, 148, 148};   // resident CTAs of the constructor in each tier
    int rf_blocks = 148;                     // resident CTAs of the refit
    int group_events = 0;                    // host-input batches: events per group (0 = automatic)
    std::vector<Batch*> slots;               // groups in flight; slots[0] always exists
    // the last call
    tpc_counters counters;
    bool have_result = false;
    bool one_group = false;                  // the last call ran as one group of device-input events (inject / resume)
    const tpc_event_in* last_in = nullptr;   // its events
    int n_events = 0;
    std::vector<int> ev_slot, ev_local;      // where the intermediates of each event are (-1: overwritten since)
    Buf<int32_t> h_o_i[kOutI], h_o_hit;          // host-input calls: the outputs of all groups, pinned
    Buf<float> h_o_f[kOutF];
    bool profiling = false;
    bool graphs = true;                      // replay the launch sequence as a CUDA graph (off while per-stage times are taken)
    float stage_ms[TPC_N_STAGES] = {};
    // tpc_submit_events / tpc_wait_events: up to three batches in flight (copy in | kernels | copy out), each with its
    // own work space, stream and outputs
    struct Async {
        Batch* b = nullptr;
        bool busy = false;
        Buf<int32_t> h_o_i[kOutI], h_o_hit;      // host inputs: this ticket's outputs, pinned
        Buf<float> h_o_f[kOutF];
        Buf<int32_t> d_o_i[kOutI], d_o_hit;      // device inputs: this ticket's outputs (swapped with the batch's at wait,
        Buf<float> d_o_f[kOutF];                 // so that the batch's next run does not write over them)
    } async[kAsync];
    int last_ticket = -1;                    // the batch submitted last (the next one's kernels queue behind its kernels)

    tpc_tracker() {
        for (auto& a : async) {
            a.h_o_hit.host = true;
            for (auto& b : a.h_o_i) b.host = true;
            for (auto& b : a.h_o_f) b.host = true;
        }
        h_o_hit.host = true;
        for (auto& b : h_o_i) b.host = true;
        for (auto& b : h_o_f) b.host = true;
        memset(&counters, 0, sizeof counters);
    }
    void sync_all() {
        for (auto s : own_streams) cudaStreamSynchronize(s);
        if (user_stream) cudaStreamSynchronize(user_stream);
        for (auto& a : async) if (a.b) cudaStreamSynchronize(a.b->stream);
    }
    void free_all() {
        for (auto* b : slots) { b->free_all(); delete b; }
        slots.clear();
        for (auto& a : async) {
            if (a.b) { cudaStreamSynchronize(a.b->stream); a.b->free_all(); cudaStreamDestroy(a.b->stream); delete a.b; a.b = nullptr; }
            a.h_o_hit.release(); a.d_o_hit.release();
            for (auto& b : a.h_o_i) b.release();
            for (auto& b : a.h_o_f) b.release();
            for (auto& b : a.d_o_i) b.release();
            for (auto& b : a.d_o_f) b.release();
        }
        for (auto s : own_streams) cudaStreamDestroy(s);
        own_streams.clear();
        h_o_hit.release();
        for (auto& b : h_o_i) b.release();
        for (auto& b : h_o_f) b.release();
    }
};

namespace {

int tab_stride(int n_rows) { return (n_rows + 31) & ~31; }

int reserve_batch(const tpc_tracker* tr, Batch* t, int n_events, int64_t N, int64_t S_cap) {
    const int64_t nb = (int64_t)n_events * tr->c.n_sectors * tr->c.n_rows;
    const size_t n = (size_t)std::max<int64_t>(N, 1);
    int rc = TPC_OK;
#define RS(b, k) if ((rc = t->b.reserve(k)) != TPC_OK) return rc
    RS(sec_off, (size_t)n_events * (tr->c.n_sectors + 1)); RS(h_sec_off, (size_t)n_events * (tr->c.n_sectors + 1));
    RS(ev_src, n_events); RS(h_ev_src, n_events);
    RS(bin_count, nb + 1); RS(bin_start, nb + 1); RS(seed_count, nb + 1); RS(seed_start, nb + 1);
    RS(slot, n); RS(thit, n); RS(tidx, n); RS(shit, n); RS(sorig, n);
    RS(desc, nb); RS(cells, (size_t)kCellsPerHit * n + (size_t)nb * kCellPad + 64);
    RS(link_up, n); RS(link_dn, n); RS(clink_up, n); RS(clink_dn, n); RS(owner, n);
    RS(seeds, S_cap); RS(seed_bin, S_cap); RS(tl_rows, S_cap); RS(tl_par, 6 * (size_t)S_cap);
    RS(tl_tab, (size_t)S_cap * tab_stride(tr->c.n_rows));
    RS(seed_rec, S_cap); RS(tl_up, S_cap); RS(dn_rec, S_cap); RS(kf_park, S_cap); RS(dn_count, nb + 1); RS(dn_start, nb + 1); RS(dn_fill, nb + 1);
    RS(tl_nown, S_cap + 1); RS(tl_keep, S_cap + 1); RS(tl_cnt, (size_t)t->sel_C * S_cap); RS(trk_scan, S_cap + 2); RS(hit_scan, S_cap + 2);
    RS(ev_off_d, 2 * ((size_t)n_events + 1)); RS(h_ev_off, 2 * ((size_t)n_events + 1));
    RS(scratch, (size_t)std::max<int64_t>(nb, S_cap) / kScanTile + 8);   // scans: tile counter + status words
    RS(cnt, CNT_N); RS(h_cnt, CNT_N); RS(kf_cursor, kNCursors); RS(h_nseeds, 1);
    {   // output arrays: only those that this tracker's parameters fill
        const int nI = tr->c.p.merge ? kOutI : kOutI_plain, nF = tr->c.p.merge ? kOutF : tr->c.p.refit ? kOutF_refit : kOutF_plain;
        for (int k = 0; k < nI; k++) RS(o_i[k], S_cap);
        for (int k = 0; k < nF; k++) RS(o_f[k], S_cap);
    }
    if (tr->c.p.refit) { RS(trk_rows, S_cap); RS(trk_task, S_cap); }
    if (tr->c.p.merge) { RS(mg_next, S_cap); RS(mg_prev, S_cap); RS(mg_list, S_cap); }
    RS(o_hit, n);
    if (tr->c.p.refit) { RS(o_hit_yz, n); RS(o_hit_row, n); RS(trk_hit0, S_cap); }
#undef RS
    t->S_cap = S_cap;
    return TPC_OK;
}

size_t ct_smem_bytes(int tier) {   // CtSmem, the shared-memory state slots, the stack of free slots
    const size_t b = sizeof(CtSmem) + (size_t)kCtWords * 4 * (size_t)kCtCapSmem[tier] + 2 * (size_t)(kCtCapSmem[tier] + kCtCapSpill[tier]);
    return (b + 127) & ~(size_t)127;
}

int64_t default_seed_cap(int64_t N) { return std::max<int64_t>(N / 8 + 4096, 4096); }

int validate(const tpc_tracker* t, int n, const tpc_event_in* in) {
    if (!t || !in || n < 1) { set_err("null tracker / events or n < 1"); return TPC_ERR_ARG; }
    const int ns = t->c.n_sectors;
    for (int e = 0; e < n; e++) {
        const tpc_event_in& ev = in[e];
        if (ev.n_clusters < 0 || !ev.sector_offset) { set_err("event %d: bad n_clusters / sector_offset", e); return TPC_ERR_ARG; }
        if (ev.mem_space != in[0].mem_space || (ev.mem_space != 0 && ev.mem_space != 1)) {
            set_err("event %d: mem_space must be 0 or 1 and the same for the whole batch", e);
            return TPC_ERR_ARG;
        }
        if (ev.n_clusters > 0 && (!ev.y || !ev.z || !ev.row)) { set_err("event %d: null cluster arrays", e); return TPC_ERR_ARG; }
        if (ev.sector_offset[0] != 0 || ev.sector_offset[ns] != ev.n_clusters) {
            set_err("event %d: sector_offset must run from 0 to n_clusters", e);
            return TPC_ERR_ARG;
        }
        for (int s = 0; s < ns; s++)
            if (ev.sector_offset[s + 1] < ev.sector_offset[s]) { set_err("event %d: sector_offset decreases", e); return TPC_ERR_ARG; }
    }
    return TPC_OK;
}

// launch K1..K6 for the staged group; counts launches
// launch the stages from `from` on (1 = K1 ... 6 = K6; TPC_STAGE_*) for the staged group; counts launches
int launch_all(const tpc_tracker* tr, Batch* t, int from = 1) {
    const View& v = t->v;
    const Const& c = tr->c;
    cudaStream_t st = t->stream;
    const int ns = c.n_sectors, nr = c.n_rows;
    const int nb = v.n_bins;
    int64_t L = 0;
    if (from <= 1) CK(cudaMemsetAsync(v.bin_count, 0, sizeof(int32_t) * (nb + 1), st));
    CK(cudaMemsetAsync(v.cnt, 0, sizeof(unsigned long long) * CNT_N, st));
    CK(cudaMemsetAsync(v.kf_cursor, 0, sizeof(unsigned long long) * kNCursors, st));
    auto mark = [&](int k) { if (tr->profiling) cudaEventRecord(t->evt[k], st); };
    mark(0);
    int maxn = 0;
    for (int e = 0; e < t->n_events; e++) maxn = std::max(maxn, t->ev_n[e]);
    if (from <= 1) {
        if (maxn > 0) {
            dim3 g((maxn + kCountChunk - 1) / kCountChunk, t->n_events);
            k_count<<<g, 256, 0, st>>>(v, c, ns, nr); L++;
        }
        L += scan_exclusive(v.bin_count, v.bin_start, nb, t->scratch.p, st);
        if (maxn > 0) {
            dim3 g((maxn + kScatterChunk - 1) / kScatterChunk, t->n_events);
            k_scatter<<<g, 256, 0, st>>>(v, ns, nr); L++;
        }
        k_sort_row<true><<<nb, kSortThreads, 0, st>>>(v); L++;
        k_sort_row<false><<<std::min(nb, 7 * tr->sm_count), kSortThreads, 0, st>>>(v); L++;
    }
    mark(1);
    if (from <= 2) { k_neighbours<<<nb, kNfThreads, 0, st>>>(v, c); L++; }
    mark(2);
    if (from <= 4) {
        if (from <= 3) k_clean<true><<<nb, kCleanThreads, 0, st>>>(v);
        else k_clean<false><<<nb, kCleanThreads, 0, st>>>(v);   // start hits of the cleaned links as they stand
        L++;
        L += scan_exclusive(v.seed_count, v.seed_start, nb, t->scratch.p, st);
        k_seeds<<<(nb + kSeedWarps - 1) / kSeedWarps, kSeedThreads, 0, st>>>(v, c); L++;
    }
    mark(3);
    if (from <= 5) {   // K5: one CTA per sector task, up sweep then down sweep (kf_construct.cuh)
        const int tier = t->ct_tier;
        const int grid = std::max(1, std::min(tr->ct_blocks[tier], v.n_tasks));
        if (tier == 0) TPC_K5_TIER0<<<grid, ct_threads(kCtWarps), ct_smem_bytes(tier), st>>>(v, c, kCtCapSpill[tier], t->ct_spill.p);
        else if (tier == 1) TPC_K5_TIER1<<<grid, ct_threads(kCtWarpsWide), ct_smem_bytes(tier), st>>>(v, c, kCtCapSpill[tier], t->ct_spill.p);
        else TPC_K5_TIER2<<<grid, ct_threads(kCtWarpsWide), ct_smem_bytes(tier), st>>>(v, c, kCtCapSpill[tier], t->ct_spill.p);
        L++;
    }
    mark(4);
    // K6: claims + owned counts per (task, chunk) in shared memory, keep flags, scans, output
    const int sel_grid = v.n_tasks * v.sel_C;
    CK(cudaMemsetAsync(v.tl_cnt, 0, sizeof(int32_t) * (size_t)v.sel_C * t->S_cap, st));
    k_select_claim<<<sel_grid, kSelCtaThreads, kSelCap * sizeof(uint32_t), st>>>(v, c); L++;
    k_select_keep<<<(int)((t->S_cap + 1 + 255) / 256), 256, 0, st>>>(v, c.p.min_track_hits); L++;
    L += scan_exclusive(v.tl_keep, v.trk_scan, (int)t->S_cap, t->scratch.p, st);
    L += scan_exclusive(v.tl_nown, v.hit_scan, (int)t->S_cap, t->scratch.p, st);
    k_event_offsets<<<(t->n_events + 1 + 63) / 64, 64, 0, st>>>(v, ns * nr); L++;
    k_select_write<<<sel_grid, kSelCtaThreads, kSelCap * sizeof(uint32_t), st>>>(v, c); L++;
    mark(5);
    if (c.p.merge) {   // the (task, row) counters of the down sweep are free again: K7 counts the refitted tracks there
        CK(cudaMemsetAsync(v.dn_count, 0, sizeof(int32_t) * (nb + 1), st));
        CK(cudaMemsetAsync(v.dn_fill, 0, sizeof(int32_t) * (nb + 1), st));
    }
    if (c.p.refit) { k_refit<<<tr->rf_blocks, kRfThreads, 0, st>>>(v, c); L++; }
    if (c.p.merge) {   // the track count is on the device: grids cover the start-hit capacity
        const int g = (int)((t->S_cap + 127) / 128);
        L += scan_exclusive(v.dn_count, v.dn_start, nb, t->scratch.p, st);
        k_merge_scatter<<<g, 128, 0, st>>>(v, nr, t->mg_list.p, t->mg_prev.p); L++;
        k_merge_pairs<<<g, 128, 0, st>>>(v, c, t->mg_list.p, t->mg_next.p, t->mg_prev.p); L++;
        k_merge_mutual<<<g, 128, 0, st>>>(v, c, t->mg_next.p, t->mg_prev.p); L++;
        k_merge_chain<<<g, 128, 0, st>>>(v, ns); L++;
        k_global_prep<<<g, kGfThreads, 0, st>>>(v, t->mg_list.p); L++;               // O10: the chains' first segments ...
        k_global_fit<<<tr->rf_blocks, kGfThreads, 0, st>>>(v, c, t->mg_list.p); L++;   // ... and their fits
    }
    mark(6);
    CK(cudaGetLastError());
    t->counters.n_kernel_launches += L;
    return TPC_OK;
}

// The same launches through a CUDA graph: captured once per shape of the group (every pointer, size and grid the
// launches bake in is part of the key), replayed afterwards -- one submission instead of ~25 (15 kernels, 10 memsets).
int launch_graphed(const tpc_tracker* tr, Batch* t) {
    // the key is built and compared as raw bytes: cleared first, members copied with memcpy (padding stays zero; the View
    // of a Batch was cleared at construction and is only ever assigned member by member)
    Batch::GraphKey key;
    memset(&key, 0, sizeof key);
    memcpy(&key.v, &t->v, sizeof(View));
    key.tier = t->ct_tier; key.n_events = t->n_events; key.S_cap = t->S_cap; key.spill = t->ct_spill.p;
    for (int e = 0; e < t->n_events; e++) key.maxn = std::max(key.maxn, t->ev_n[e]);
    int k = -1;
    for (int i = 0; i < Batch::kGraphs; i++)
        if (t->gexec[i] && memcmp(&key, &t->gkey[i], sizeof key) == 0) k = i;
    if (k < 0) {
        k = t->graph_victim;
        t->graph_victim = (k + 1) % Batch::kGraphs;
        if (t->gexec[k]) { cudaGraphExecDestroy(t->gexec[k]); t->gexec[k] = nullptr; }
        cudaGraph_t g = nullptr;
        CK(cudaStreamBeginCapture(t->stream, cudaStreamCaptureModeThreadLocal));
        const int64_t before = t->counters.n_kernel_launches;
        const int rc = launch_all(tr, t);
        const cudaError_t e = cudaStreamEndCapture(t->stream, &g);
        t->graph_launches[k] = t->counters.n_kernel_launches - before;
        t->counters.n_kernel_launches = before;
        if (rc != TPC_OK) { if (g) cudaGraphDestroy(g); return rc; }
        if (e != cudaSuccess || !g) { set_err("graph capture failed: %s", cudaGetErrorString(e)); return TPC_ERR_CUDA; }
        const cudaError_t ei = cudaGraphInstantiate(&t->gexec[k], g, 0);
        cudaGraphDestroy(g);
        if (ei != cudaSuccess) { t->gexec[k] = nullptr; set_err("graph instantiation failed: %s", cudaGetErrorString(ei)); return TPC_ERR_CUDA; }
        memcpy(&t->gkey[k], &key, sizeof key);
    }
    CK(cudaGraphLaunch(t->gexec[k], t->stream));
    t->counters.n_kernel_launches += t->graph_launches[k];
    return TPC_OK;
}

// Enqueue one group of events on its slot's stream: input copies (host inputs), K1..K6, the counters' way back.
// Nothing here waits for the device.
int batch_begin(const tpc_tracker* tr, Batch* t, int first_event, int n, const tpc_event_in* in, int64_t S_cap, bool copy_inputs) {
    const int ns = tr->c.n_sectors, nr = tr->c.n_rows;
    int rc;
    int64_t N = 0;
    t->ev_n.assign(n, 0); t->ev_off.assign(n + 1, 0);
    for (int e = 0; e < n; e++) { t->ev_n[e] = in[e].n_clusters; t->ev_off[e] = (int32_t)N; N += in[e].n_clusters; }
    t->ev_off[n] = (int32_t)N;
    if (N > 0x7fff0000ll) { set_err("a group of events holds more than 2^31 clusters"); return TPC_ERR_CAPACITY; }
    t->host_in = in[0].mem_space == 0;
    t->in = in; t->first_event = first_event;
    cudaStream_t st = t->stream;
    S_cap = std::max<int64_t>(std::max<int64_t>(t->S_cap, S_cap), default_seed_cap(N));
    {   // selector: chunks per sector task so that a chunk's owner words fit the shared memory (a chunk holds at
        // most its share of the task's hits plus one pad row)
        int64_t max_task = 0;
        for (int e = 0; e < n; e++)
            for (int s = 0; s < ns; s++)
                max_task = std::max<int64_t>(max_task, in[e].sector_offset[s + 1] - in[e].sector_offset[s]);
        const int64_t room = kSelCap - TPC_MAX_ROW_HITS - 1;
        t->sel_C = (int)std::max<int64_t>(1, (max_task + room - 1) / room);   // of THIS group (tl_cnt only grows)
    }
    if ((rc = reserve_batch(tr, t, n, N, S_cap)) != TPC_OK) return rc;
    if (t->host_in) {
        const size_t nn = (size_t)std::max<int64_t>(N, 1);
        if ((rc = t->in_y.reserve(nn)) != TPC_OK || (rc = t->in_z.reserve(nn)) != TPC_OK || (rc = t->in_row.reserve(nn)) != TPC_OK)
            return rc;
        if (tr->c.p.checked && (rc = t->in_x.reserve(nn)) != TPC_OK) return rc;
    }
    // the event table and the sector offsets
    for (int e = 0; e < n; e++) {
        EventSrc& s = t->h_ev_src.p[e];
        s.n = in[e].n_clusters; s.off = t->ev_off[e];
        s.x = nullptr;
        if (t->host_in) {
            s.y = t->in_y.p + s.off; s.z = t->in_z.p + s.off; s.row = t->in_row.p + s.off;
            if (tr->c.p.checked && in[e].x) {
                s.x = t->in_x.p + s.off;
                if (copy_inputs && s.n > 0) CK(cudaMemcpyAsync(t->in_x.p + s.off, in[e].x, sizeof(float) * s.n, cudaMemcpyHostToDevice, st));
            }
            if (copy_inputs && s.n > 0) {
                CK(cudaMemcpyAsync(t->in_y.p + s.off, in[e].y, sizeof(float) * s.n, cudaMemcpyHostToDevice, st));
                CK(cudaMemcpyAsync(t->in_z.p + s.off, in[e].z, sizeof(float) * s.n, cudaMemcpyHostToDevice, st));
                CK(cudaMemcpyAsync(t->in_row.p + s.off, in[e].row, sizeof(int32_t) * s.n, cudaMemcpyHostToDevice, st));
            }
        } else {
            s.x = tr->c.p.checked ? in[e].x : nullptr; s.y = in[e].y; s.z = in[e].z; s.row = in[e].row;
        }
        memcpy(t->h_sec_off.p + (size_t)e * (ns + 1), in[e].sector_offset, sizeof(int32_t) * (ns + 1));
    }
    CK(cudaMemcpyAsync(t->ev_src.p, t->h_ev_src.p, sizeof(EventSrc) * n, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(t->sec_off.p, t->h_sec_off.p, sizeof(int32_t) * (size_t)n * (ns + 1), cudaMemcpyHostToDevice, st));

    View& v = t->v;
    v.n_events = n; v.n_tasks = n * ns; v.n_bins = n * ns * nr; v.N = (int32_t)N;
    v.ev = t->ev_src.p; v.sec_off = t->sec_off.p;
    v.bin_count = t->bin_count.p; v.bin_start = t->bin_start.p; v.slot = t->slot.p;
    v.thit = t->thit.p; v.tidx = t->tidx.p; v.shit = t->shit.p; v.sorig = t->sorig.p;
    v.desc = t->desc.p; v.cells = t->cells.p;
    v.link_up = t->link_up.p; v.link_dn = t->link_dn.p; v.clink_up = t->clink_up.p; v.clink_dn = t->clink_dn.p;
    v.seed_count = t->seed_count.p; v.seed_start = t->seed_start.p; v.seeds = t->seeds.p; v.seed_bin = t->seed_bin.p;
    v.S_cap = (int32_t)t->S_cap;
    v.tl_tab = t->tl_tab.p; v.tab_stride = tab_stride(nr); v.tl_rows = t->tl_rows.p; v.tl_par = t->tl_par.p;
    v.owner = t->owner.p; v.tl_nown = t->tl_nown.p; v.tl_keep = t->tl_keep.p; v.tl_cnt = t->tl_cnt.p; v.sel_C = t->sel_C;
    v.trk_scan = t->trk_scan.p; v.hit_scan = t->hit_scan.p; v.ev_off = t->ev_off_d.p;
    v.o_sector = t->o_i[0].p; v.o_first_hit = t->o_i[1].p; v.o_n_hits = t->o_i[2].p; v.o_ndf = t->o_i[3].p;
    v.o_hit_idx = t->o_hit.p;
    v.o_x = t->o_f[0].p; v.o_y = t->o_f[1].p; v.o_z = t->o_f[2].p; v.o_sinphi = t->o_f[3].p;
    v.o_tgl = t->o_f[4].p; v.o_qpt = t->o_f[5].p; v.o_chi2 = t->o_f[6].p;
    v.o_xo = t->o_f[7].p; v.o_yo = t->o_f[8].p; v.o_zo = t->o_f[9].p; v.o_so = t->o_f[10].p; v.o_to = t->o_f[11].p; v.o_qo = t->o_f[12].p;
    v.o_gndf = t->o_i[7].p; v.o_gnhits = t->o_i[8].p; v.o_gsector = t->o_i[9].p;
    v.o_gx = t->o_f[13].p; v.o_gy = t->o_f[14].p; v.o_gz = t->o_f[15].p; v.o_gs = t->o_f[16].p; v.o_gt = t->o_f[17].p;
    v.o_gq = t->o_f[18].p; v.o_gchi2 = t->o_f[19].p;
    v.o_next = t->o_i[4].p; v.o_prev = t->o_i[5].p; v.o_global = t->o_i[6].p; v.trk_rows = t->trk_rows.p; v.trk_task = t->trk_task.p;
    v.cnt = t->cnt.p; v.kf_cursor = t->kf_cursor.p;
    v.o_hit_yz = t->o_hit_yz.p; v.o_hit_row = t->o_hit_row.p; v.trk_hit0 = t->trk_hit0.p;
    v.seed_rec = t->seed_rec.p; v.tl_up = t->tl_up.p; v.dn_rec = t->dn_rec.p; v.kf_park = t->kf_park.p;
    v.dn_count = t->dn_count.p; v.dn_start = t->dn_start.p; v.dn_fill = t->dn_fill.p;
    t->ct_tier = tr->ct_tier;   // what earlier overflows have taught the tracker
    // few sector tasks (a single event): one wide CTA per SM serves a task in one round per row (measured on one
    // central event: K5 1.46 ms against 2.06 ms with the two-CTAs-per-SM tier; on 16 events 5.83 against 4.72 ms)
    if (n * ns <= tr->sm_count) t->ct_tier = std::max(t->ct_tier, 1);
    if (kCtCapSpill[t->ct_tier] > 0) {   // slots in global memory for every resident CTA (allocated once, on the way up)
        if ((rc = t->ct_spill.reserve((size_t)tr->ct_blocks[t->ct_tier] * kCtWords * kCtCapSpill[t->ct_tier])) != TPC_OK) return rc;
    }
    t->n_events = n; t->N = N;
    if (tr->profiling)
        for (auto& e : t->evt)
            if (!e) CK(cudaEventCreate(&e));

    // submit / wait pipeline: the input copies above run beside the other batch's kernels, the kernels behind them
    if (t->wait_for) CK(cudaStreamWaitEvent(st, t->wait_for, 0));
    if ((rc = (tr->graphs && !tr->profiling) ? launch_graphed(tr, t) : launch_all(tr, t)) != TPC_OK) return rc;
    if (t->kernels_done) CK(cudaEventRecord(t->kernels_done, st));
    CK(cudaMemcpyAsync(t->h_cnt.p, v.cnt, sizeof(unsigned long long) * CNT_N, cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(t->h_ev_off.p, v.ev_off, sizeof(int32_t) * 2 * (n + 1), cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(t->h_nseeds.p, v.seed_start + v.n_bins, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    return TPC_OK;
}

// Wait for the group, check what the kernels reported, grow the tracklet pools and run again if they overflowed.
int batch_finish(const tpc_tracker* tr, Batch* t) {
    const int nr = tr->c.n_rows;
    for (int attempt = 0;; attempt++) {
        CK(cudaStreamSynchronize(t->stream));
        if (tr->profiling)
            for (int k = 0; k < TPC_N_STAGES; k++) cudaEventElapsedTime(&t->stage_ms[k], t->evt[k], t->evt[k + 1]);
        const unsigned err = (unsigned)(t->h_cnt.p[CNT_ERR] & 0xffffffffu);
        const int32_t n_seeds = t->h_nseeds.p[0];
        if (err & kErrBadRow) { set_err("a cluster has row outside [0,%d)", nr); return TPC_ERR_ARG; }
        if (err & kErrBadInput) { set_err("checked mode: a cluster has a non-finite y or z, or an x more than 1e-3 cm off row_x[row]"); return TPC_ERR_ARG; }
        if (err & kErrHang) { set_err("the constructor lost a shared-memory pipeline signal"); return TPC_ERR_CUDA; }
        if (err & kErrSelCapacity) { set_err("selector: a chunk of pad rows exceeds the shared-memory owner table"); return TPC_ERR_CAPACITY; }
        if (err & kErrRowCapacity) {
            set_err("more than %d clusters in one (sector,row)", TPC_MAX_ROW_HITS);
            return TPC_ERR_CAPACITY;
        }
        const bool slots = (err & kErrSlotCapacity) != 0;
        if (slots && t->ct_tier >= kCtTiers - 1) {
            set_err("more than %d tracklets under way at once in one sector task", kCtCapMax);
            return TPC_ERR_CAPACITY;
        }
        if (slots || (err & kErrSeedCapacity) || n_seeds > t->S_cap) {
            if (attempt >= 4) { set_err("tracklet pool could not be grown"); return TPC_ERR_CAPACITY; }
            t->counters.n_retries++;
            if (slots) { t->ct_tier++; const_cast<tpc_tracker*>(tr)->ct_tier = t->ct_tier; }   // sticky: the tracker stays in the higher tier
            int rc = batch_begin(tr, t, t->first_event, t->n_events, t->in, std::max<int64_t>(t->S_cap, (int64_t)n_seeds + n_seeds / 8 + 1024), false);
            if (rc != TPC_OK) return rc;
            continue;
        }
        t->counters.n_events = t->n_events; t->counters.n_clusters = t->N;
        t->counters.n_links = (int64_t)t->h_cnt.p[CNT_LINKS];
        t->counters.n_seeds = n_seeds;
        t->counters.n_row_visits = (int64_t)t->h_cnt.p[CNT_ROW_VISITS];
        t->counters.n_tracklet_hits = (int64_t)t->h_cnt.p[CNT_TL_HITS];
        t->counters.n_tracks = (int64_t)t->h_cnt.p[CNT_TRACKS];
        t->counters.n_track_hits = (int64_t)t->h_cnt.p[CNT_TRACK_HITS];
        t->counters.n_updates = (int64_t)t->h_cnt.p[CNT_UPDATES];
        t->counters.n_refit_visits = (int64_t)t->h_cnt.p[CNT_REFIT_VISITS];
        t->counters.n_tracklets = (int64_t)t->h_cnt.p[CNT_TRACKLETS];
        return TPC_OK;
    }
}

Batch* get_slot(tpc_tracker* t, int k) {
    while ((int)t->slots.size() <= k) {
        cudaStream_t s = nullptr;
        if (cudaStreamCreateWithFlags(&s, cudaStreamNonBlocking) != cudaSuccess) { set_err("cudaStreamCreate failed"); return nullptr; }
        t->own_streams.push_back(s);
        Batch* b = new Batch;
        b->stream = s;
        t->slots.push_back(b);
    }
    return t->slots[k];
}

// pinned output array of a host-input call: grow, keeping what earlier groups have written
template <class T> int grow_keep(tpc_tracker* t, Buf<T>& b, size_t need, size_t keep, size_t hint) {
    if (need <= b.cap) return TPC_OK;
    t->sync_all();   // copies into the old array may be in flight
    Buf<T> nb; nb.host = true;
    int rc = nb.reserve(std::max(need, hint));
    if (rc != TPC_OK) return rc;
    if (keep) memcpy(nb.p, b.p, keep * sizeof(T));
    b.release();
    b = nb;
    return TPC_OK;
}

void add_counters(tpc_counters& a, const tpc_counters& b) {
    a.n_events += b.n_events; a.n_clusters += b.n_clusters; a.n_links += b.n_links; a.n_seeds += b.n_seeds;
    a.n_row_visits += b.n_row_visits; a.n_tracklet_hits += b.n_tracklet_hits; a.n_tracks += b.n_tracks;
    a.n_track_hits += b.n_track_hits; a.n_kernel_launches += b.n_kernel_launches; a.n_retries += b.n_retries; a.n_updates += b.n_updates; a.n_refit_visits += b.n_refit_visits; a.n_tracklets += b.n_tracklets;
}

}  // namespace

extern "C" {

void tpc_default_params(tpc_params* p) {
    if (!p) return;
    p->link_step = 1;
    p->nf_slope_y = 1.5f; p->nf_slope_z = 2.0f; p->nf_w0 = 0.3f; p->nf_dmax = 0.25f;
    p->sin_max = 0.95f;
    p->var_s = 0.25f; p->var_t = 1.0f; p->var_q = 100.0f;
    p->chi2_link = 25.0f; p->chi2_ext = 16.0f;
    p->win_nsigma = 4.0f; p->win_min = 0.3f; p->win_max = 3.0f;
    p->max_gap = 5; p->edge_margin = 1.0f;
    p->min_tracklet_hits = 10; p->min_track_hits = 10;
    p->refit = 0;
    p->merge = 0; p->merge_dy = 1.0f; p->merge_dz = 1.0f; p->merge_ds = 0.05f; p->merge_dt = 0.05f; p->merge_max_gap = 6;
    p->seed_dedup = 1;
    p->checked = 0;
}

const char* tpc_status_string(int s) {
    switch (s) {
        case TPC_OK: return "ok";
        case TPC_ERR_ARG: return "bad argument";
        case TPC_ERR_GEOMETRY: return "bad geometry";
        case TPC_ERR_CAPACITY: return "capacity exceeded";
        case TPC_ERR_CUDA: return "CUDA error";
        default: return "unknown status";
    }
}

const char* tpc_last_error(void) { return g_err.c_str(); }

tpc_tracker* tpc_tracker_create_ex(const tpc_geometry* g, float bz, const tpc_params* params, int32_t max_events,
                                   int64_t max_clusters) {
    if (!g || !g->row_x) { set_err("null geometry"); return nullptr; }
    if (g->n_rows < 3 || g->n_rows > TPC_MAX_ROWS || g->n_sectors < 1 || g->n_sectors > 64) {
        set_err("geometry: n_rows must be in [3,%d], n_sectors in [1,64]", TPC_MAX_ROWS);
        return nullptr;
    }
    for (int r = 1; r < g->n_rows; r++)
        if (!(g->row_x[r] > g->row_x[r - 1])) { set_err("geometry: row_x must be strictly increasing"); return nullptr; }
    if (!(g->sigma_y > 0.f) || !(g->sigma_z > 0.f) || !(g->tan_half_angle > 0.f)) {
        set_err("geometry: sigma_y, sigma_z, tan_half_angle must be positive");
        return nullptr;
    }
    tpc_params p;
    if (params) p = *params; else tpc_default_params(&p);
    if (p.link_step < 1 || p.link_step > 2 || p.min_tracklet_hits < 1 || p.min_track_hits < 1 || p.max_gap < 0 || p.max_gap > 60 ||
        p.seed_dedup < 0 || p.seed_dedup > 1 || p.refit < 0 || p.refit > 1 || p.merge < 0 || p.merge > 1 ||
        p.checked < 0 || p.checked > 1 || (p.merge && !p.refit) || p.merge_max_gap < 0 || !(p.merge_dy > 0.f) || !(p.merge_dz > 0.f) || !(p.merge_ds > 0.f) || !(p.merge_dt > 0.f)) {
        set_err("params: link_step must be 1 or 2, minimum hit counts >= 1, max_gap in [0,60], seed_dedup 0 or 1, refit 0 or 1, merge 0 or 1 (needs refit) with positive tolerances");
        return nullptr;
    }
    int dev = 0, ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        set_err("no CUDA device: libtpctrack has no CPU fallback");
        cudaGetLastError();
        return nullptr;
    }
    cudaGetDevice(&dev);
    tpc_tracker* t = new tpc_tracker;
    memset(&t->c, 0, sizeof t->c);
    for (int r = 0; r < g->n_rows; r++) t->c.row_x[r] = g->row_x[r];
    t->c.n_sectors = g->n_sectors; t->c.n_rows = g->n_rows;
    t->c.tan_half_angle = g->tan_half_angle;
    t->c.sigma_y2 = g->sigma_y * g->sigma_y; t->c.sigma_z2 = g->sigma_z * g->sigma_z;
    t->c.kB = -1.f * (0.00299792458f * bz);  // curvature = kB * q/pT, DESIGN.md "Conventions"
    t->c.p = p;
    {   // O9: angle between neighbouring sectors, rounded once to float
        const double step = 2.0 * 3.14159265358979323846 / (double)std::max(g->n_sectors / 2, 1);
        t->c.merge_cd = (float)cos(step); t->c.merge_sd = (float)sin(step);
    }
    if (g->sector_alpha) t->sector_alpha.assign(g->sector_alpha, g->sector_alpha + g->n_sectors);
    cudaDeviceGetAttribute(&t->sm_count, cudaDevAttrMultiProcessorCount, dev);
    {   // persistent constructor grid: as many CTAs as are resident at once, for both slot counts
        int per_sm = 0;
        size_t most = 0;
        for (int k = 0; k < kCtTiers; k++) most = std::max(most, ct_smem_bytes(k));
        if (cudaFuncSetAttribute(TPC_K5_TIER0, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ct_smem_bytes(0)) != cudaSuccess ||
            cudaFuncSetAttribute(TPC_K5_TIER1, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)most) != cudaSuccess ||
            cudaFuncSetAttribute(TPC_K5_TIER2, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)most) != cudaSuccess) {
            set_err("k_construct: %zu bytes of shared memory cannot be configured: %s", most, cudaGetErrorString(cudaGetLastError()));
            delete t;
            return nullptr;
        }
        for (int k = 0; k < kCtTiers; k++) {
            const cudaError_t e = k == 0
                ? cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, TPC_K5_TIER0, ct_threads(kCtWarps), ct_smem_bytes(k))
                : cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, TPC_K5_TIER2, ct_threads(kCtWarpsWide), ct_smem_bytes(k));
            if (e != cudaSuccess || per_sm < 1) {
                set_err("k_construct cannot be configured: %s", cudaGetErrorString(cudaGetLastError()));
                delete t;
                return nullptr;
            }
            t->ct_blocks[k] = t->sm_count * per_sm;
            if (getenv("TPCTRACK_VERBOSE")) fprintf(stderr, "[tpctrack] K5 tier %d: %d CTAs per SM, %zu bytes of shared memory\n", k, per_sm, ct_smem_bytes(k));
        }
        if (!p.seed_dedup) t->ct_tier = 1;   // ~3x the tracklets under way
        if (const char* se = getenv("TPCTRACK_CT_TIER")) t->ct_tier = std::max(0, std::min(atoi(se), kCtTiers - 1));
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_refit, kRfThreads, 0) != cudaSuccess || per_sm < 1) per_sm = 1;
        t->rf_blocks = t->sm_count * per_sm;
        if (cudaFuncSetAttribute(k_select_claim, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(kSelCap * sizeof(uint32_t))) != cudaSuccess ||
            cudaFuncSetAttribute(k_select_write, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(kSelCap * sizeof(uint32_t))) != cudaSuccess) {
            set_err("the selector's shared memory cannot be configured: %s", cudaGetErrorString(cudaGetLastError()));
            delete t;
            return nullptr;
        }
    }
    if (const char* ge = getenv("TPCTRACK_GROUP_EVENTS")) t->group_events = atoi(ge);
    if (const char* gg = getenv("TPCTRACK_GRAPHS")) t->graphs = atoi(gg) != 0;
    Batch* b0 = get_slot(t, 0);
    if (!b0) { t->free_all(); delete t; return nullptr; }
    if (max_events > 0 && max_clusters > 0) {
        if (reserve_batch(t, b0, max_events, max_clusters, default_seed_cap(max_clusters)) != TPC_OK) {
            t->free_all(); delete t;
            return nullptr;
        }
    }
    return t;
}

tpc_tracker* tpc_tracker_create(const tpc_geometry* g, float bz) { return tpc_tracker_create_ex(g, bz, nullptr, 0, 0); }

void tpc_tracker_destroy(tpc_tracker* t) {
    if (!t) return;
    t->sync_all();
    t->free_all();
    delete t;
}

int tpc_tracker_set_stream(tpc_tracker* t, void* s) {
    if (!t) return TPC_ERR_ARG;
    t->user_stream = (cudaStream_t)s;
    return TPC_OK;
}

int tpc_tracker_set_group_events(tpc_tracker* t, int32_t n) {
    if (!t || n < 0) return TPC_ERR_ARG;
    t->group_events = n;
    return TPC_OK;
}

int tpc_track_events(tpc_tracker* t, int32_t n, const tpc_event_in* in, tpc_event_out* out) {
    int rc = validate(t, n, in);
    if (rc != TPC_OK) return rc;
    if (!out) { set_err("null output array"); return TPC_ERR_ARG; }
    t->have_result = false;
    memset(&t->counters, 0, sizeof t->counters);
    for (float& m : t->stage_ms) m = 0.f;
    const bool host_in = in[0].mem_space == 0;
    int64_t N = 0;
    for (int e = 0; e < n; e++) N += in[e].n_clusters;

    // Groups of events.  Device inputs: one group (every launch covers the whole batch).  Host inputs: a few groups
    // on their own streams, so that the copies of one group overlap the kernels of another.
    int per_group = n;
    if (!host_in && n > 1 && t->group_events > 0) per_group = std::max(std::min<int>(t->group_events, n), (n + 3) / 4);
    if (host_in && n > 1) {
        if (t->group_events > 0) per_group = std::min<int>(t->group_events, n);
        else {
            const int want = (int)std::min<int64_t>(4, std::max<int64_t>(1, N / 2000000));   // >= ~2 M clusters per group
            per_group = (n + want - 1) / want;
        }
    }
    const int n_groups = (n + per_group - 1) / per_group;
    const int n_slots = host_in ? std::min(n_groups, 3) : n_groups;   // device inputs: outputs stay in the slots
    for (int k = 0; k < n_slots; k++)
        if (!get_slot(t, k)) return TPC_ERR_CUDA;
    for (int k = 0; k < n_slots; k++) {
        t->slots[k]->stream = (n_groups == 1 && t->user_stream) ? t->user_stream : t->own_streams[k];
        memset(&t->slots[k]->counters, 0, sizeof(tpc_counters));
    }
    t->ev_slot.assign(n, -1); t->ev_local.assign(n, 0);
    t->n_events = n;

    int64_t T_cum = 0, H_cum = 0;
    const int nI = t->c.p.merge ? kOutI : kOutI_plain, nF = t->c.p.merge ? kOutF : t->c.p.refit ? kOutF_refit : kOutF_plain;   // arrays that hold something
    std::vector<int64_t> trk_off(n + 1, 0), hit_off(n + 1, 0);   // per event, in the call's output arrays
    std::vector<const Batch*> ev_batch(n, nullptr);
    int g_issue = 0, g_done = 0;
    while (g_done < n_groups) {
        while (g_issue < n_groups && g_issue - g_done < n_slots) {
            Batch* b = t->slots[g_issue % n_slots];
            const int e0 = g_issue * per_group, ne = std::min(per_group, n - e0);
            memset(&b->counters, 0, sizeof(tpc_counters));
            if ((rc = batch_begin(t, b, e0, ne, in + e0, 0, true)) != TPC_OK) { t->sync_all(); return rc; }
            g_issue++;
        }
        Batch* b = t->slots[g_done % n_slots];
        if ((rc = batch_finish(t, b)) != TPC_OK) { t->sync_all(); return rc; }
        add_counters(t->counters, b->counters);
        if (t->profiling) for (int k = 0; k < TPC_N_STAGES; k++) t->stage_ms[k] += b->stage_ms[k];
        const int64_t T = b->counters.n_tracks, H = b->counters.n_track_hits;
        const int e0 = b->first_event, ne = b->n_events;
        const int32_t* toff = b->h_ev_off.p;
        const int32_t* hoff = b->h_ev_off.p + (ne + 1);
        for (int e = 0; e < ne; e++) {
            // host inputs: the groups' outputs are concatenated; device inputs: each group keeps its own arrays
            trk_off[e0 + e] = (host_in ? T_cum : 0) + toff[e]; hit_off[e0 + e] = (host_in ? H_cum : 0) + hoff[e];
            out[e0 + e].n_tracks = toff[e + 1] - toff[e];
            out[e0 + e].n_track_hits = hoff[e + 1] - hoff[e];
        }
        for (int e = 0; e < n; e++) if (t->ev_slot[e] == g_done % n_slots) t->ev_slot[e] = -1;   // overwritten
        for (int e = 0; e < ne; e++) { t->ev_slot[e0 + e] = g_done % n_slots; t->ev_local[e0 + e] = e; }
        if (host_in) {   // the group's tracks go behind those of the groups before it
            const size_t left = (size_t)(n_groups - g_done - 1);
            const View& v = b->v;
            const size_t needT = (size_t)std::max<int64_t>(T_cum + T, 1), hintT = needT + needT / 8 + left * (size_t)(T + T / 4);
            const size_t needH = (size_t)std::max<int64_t>(H_cum + H, 1), hintH = needH + needH / 8 + left * (size_t)(H + H / 4);
            for (int k = 0; k < nI; k++) {
                if ((rc = grow_keep(t, t->h_o_i[k], needT, (size_t)T_cum, hintT)) != TPC_OK) return rc;
                if (T) CK(cudaMemcpyAsync(t->h_o_i[k].p + T_cum, b->o_i[k].p, sizeof(int32_t) * T, cudaMemcpyDeviceToHost, b->stream));
            }
            for (int k = 0; k < nF; k++) {
                if ((rc = grow_keep(t, t->h_o_f[k], needT, (size_t)T_cum, hintT)) != TPC_OK) return rc;
                if (T) CK(cudaMemcpyAsync(t->h_o_f[k].p + T_cum, b->o_f[k].p, sizeof(float) * T, cudaMemcpyDeviceToHost, b->stream));
            }
            if ((rc = grow_keep(t, t->h_o_hit, needH, (size_t)H_cum, hintH)) != TPC_OK) return rc;
            if (H) CK(cudaMemcpyAsync(t->h_o_hit.p + H_cum, v.o_hit_idx, sizeof(int32_t) * H, cudaMemcpyDeviceToHost, b->stream));
        } else {
            for (int e = 0; e < ne; e++) ev_batch[e0 + e] = b;
        }
        T_cum += T; H_cum += H;
        g_done++;
    }
    if (host_in)
        for (int k = 0; k < n_slots; k++) CK(cudaStreamSynchronize(t->slots[k]->stream));
    for (int e = 0; e < n; e++) {
        tpc_event_out& o = out[e];
        const int32_t* oi[kOutI]; const float* of[kOutF]; const int32_t* ohit;
        int64_t a = trk_off[e], h = hit_off[e];
        if (host_in) {
            for (int k = 0; k < kOutI; k++) oi[k] = t->h_o_i[k].p;
            for (int k = 0; k < kOutF; k++) of[k] = t->h_o_f[k].p;
            ohit = t->h_o_hit.p;
        } else {
            const Batch* b = ev_batch[e];
            for (int k = 0; k < kOutI; k++) oi[k] = b->o_i[k].p;
            for (int k = 0; k < kOutF; k++) of[k] = b->o_f[k].p;
            ohit = b->v.o_hit_idx;
        }
        o.trk_sector = oi[0] + a; o.trk_first_hit = oi[1] + a; o.trk_n_hits = oi[2] + a; o.trk_ndf = oi[3] + a;
        o.trk_x = of[0] + a; o.trk_y = of[1] + a; o.trk_z = of[2] + a; o.trk_sinphi = of[3] + a; o.trk_tgl = of[4] + a;
        o.trk_qpt = of[5] + a; o.trk_chi2 = of[6] + a;
        const bool rf = t->c.p.refit != 0, mg = t->c.p.merge != 0;
        o.trk_out_x = rf ? of[7] + a : nullptr; o.trk_out_y = rf ? of[8] + a : nullptr; o.trk_out_z = rf ? of[9] + a : nullptr;
        o.trk_out_sinphi = rf ? of[10] + a : nullptr; o.trk_out_tgl = rf ? of[11] + a : nullptr;
        o.trk_out_qpt = rf ? of[12] + a : nullptr;
        o.trk_next = mg ? oi[4] + a : nullptr; o.trk_prev = mg ? oi[5] + a : nullptr; o.trk_global = mg ? oi[6] + a : nullptr;
        o.trk_g_ndf = mg ? oi[7] + a : nullptr; o.trk_g_n_hits = mg ? oi[8] + a : nullptr; o.trk_g_sector = mg ? oi[9] + a : nullptr;
        o.trk_g_x = mg ? of[13] + a : nullptr; o.trk_g_y = mg ? of[14] + a : nullptr; o.trk_g_z = mg ? of[15] + a : nullptr;
        o.trk_g_sinphi = mg ? of[16] + a : nullptr; o.trk_g_tgl = mg ? of[17] + a : nullptr; o.trk_g_qpt = mg ? of[18] + a : nullptr;
        o.trk_g_chi2 = mg ? of[19] + a : nullptr;
        o.hit_idx = ohit + h;
    }
    t->have_result = true;
    t->one_group = !host_in && n_groups == 1;
    t->last_in = in;
    return TPC_OK;
}

int tpc_submit_events(tpc_tracker* t, int32_t n, const tpc_event_in* in, int32_t* ticket) {
    int rc = validate(t, n, in);
    if (rc != TPC_OK) return rc;
    if (!ticket) { set_err("null ticket"); return TPC_ERR_ARG; }
    int k = -1;
    for (int j = 0; j < kAsync; j++) if (!t->async[j].busy) { k = j; break; }
    if (k < 0) { set_err("%d batches are in flight: wait for one first", kAsync); return TPC_ERR_ARG; }
    tpc_tracker::Async& a = t->async[k];
    if (!a.b) {
        cudaStream_t s = nullptr;
        if (cudaStreamCreateWithFlags(&s, cudaStreamNonBlocking) != cudaSuccess) { set_err("cudaStreamCreate failed"); return TPC_ERR_CUDA; }
        a.b = new Batch;
        a.b->stream = s;
        if (cudaEventCreateWithFlags(&a.b->kernels_done, cudaEventDisableTiming) != cudaSuccess) { set_err("cudaEventCreate failed"); return TPC_ERR_CUDA; }
    }
    // copy-in | kernels | copy-out pipeline: the kernels of this batch queue behind those of the batch submitted before
    // it, so that two batches never share the SMs; only the copies run beside another batch's kernels
    a.b->wait_for = nullptr;
    if (t->last_ticket >= 0 && t->last_ticket != k) {
        tpc_tracker::Async& o = t->async[t->last_ticket];
        if (o.busy && o.b) a.b->wait_for = o.b->kernels_done;
    }
    memset(&a.b->counters, 0, sizeof(tpc_counters));
    if ((rc = batch_begin(t, a.b, 0, n, in, 0, true)) != TPC_OK) { cudaStreamSynchronize(a.b->stream); return rc; }
    a.busy = true;
    t->last_ticket = k;
    *ticket = k;
    return TPC_OK;
}

int tpc_wait_events(tpc_tracker* t, int32_t ticket, tpc_event_out* out) {
    if (!t || !out || ticket < 0 || ticket >= kAsync || !t->async[ticket].busy) { set_err("no batch in flight under this ticket"); return TPC_ERR_ARG; }
    tpc_tracker::Async& a = t->async[ticket];
    Batch* b = a.b;
    a.busy = false;
    int rc = batch_finish(t, b);
    if (rc != TPC_OK) { cudaStreamSynchronize(b->stream); return rc; }
    t->counters = b->counters;
    if (t->profiling) for (int k = 0; k < TPC_N_STAGES; k++) t->stage_ms[k] = b->stage_ms[k];
    t->have_result = false;   // no intermediates for these batches
    t->one_group = false;
    const int n = b->n_events;
    const int64_t T = b->counters.n_tracks, H = b->counters.n_track_hits;
    const int nI = t->c.p.merge ? kOutI : kOutI_plain, nF = t->c.p.merge ? kOutF : t->c.p.refit ? kOutF_refit : kOutF_plain;
    const int32_t* oi[kOutI]; const float* of[kOutF]; const int32_t* ohit;
    if (b->host_in) {
        for (int k = 0; k < nI; k++) {
            if ((rc = a.h_o_i[k].reserve((size_t)std::max<int64_t>(T, 1))) != TPC_OK) return rc;
            if (T) CK(cudaMemcpyAsync(a.h_o_i[k].p, b->o_i[k].p, sizeof(int32_t) * T, cudaMemcpyDeviceToHost, b->stream));
        }
        for (int k = 0; k < nF; k++) {
            if ((rc = a.h_o_f[k].reserve((size_t)std::max<int64_t>(T, 1))) != TPC_OK) return rc;
            if (T) CK(cudaMemcpyAsync(a.h_o_f[k].p, b->o_f[k].p, sizeof(float) * T, cudaMemcpyDeviceToHost, b->stream));
        }
        if ((rc = a.h_o_hit.reserve((size_t)std::max<int64_t>(H, 1))) != TPC_OK) return rc;
        if (H) CK(cudaMemcpyAsync(a.h_o_hit.p, b->v.o_hit_idx, sizeof(int32_t) * H, cudaMemcpyDeviceToHost, b->stream));
        CK(cudaStreamSynchronize(b->stream));
        for (int k = 0; k < kOutI; k++) oi[k] = a.h_o_i[k].p;
        for (int k = 0; k < kOutF; k++) of[k] = a.h_o_f[k].p;
        ohit = a.h_o_hit.p;
    } else {
        // the ticket takes the arrays that hold this run's outputs; the batch goes on with the ticket's previous ones
        // (whose contents the caller no longer needs: they belong to the wait before last on this ticket)
        for (int k = 0; k < kOutI; k++) { std::swap(a.d_o_i[k], b->o_i[k]); oi[k] = a.d_o_i[k].p; }
        for (int k = 0; k < kOutF; k++) { std::swap(a.d_o_f[k], b->o_f[k]); of[k] = a.d_o_f[k].p; }
        std::swap(a.d_o_hit, b->o_hit);
        ohit = a.d_o_hit.p;
    }
    const int32_t* toff = b->h_ev_off.p;
    const int32_t* hoff = b->h_ev_off.p + (n + 1);
    const bool rf = t->c.p.refit != 0, mg = t->c.p.merge != 0;
    for (int e = 0; e < n; e++) {
        tpc_event_out& o = out[e];
        const int64_t at = toff[e], ah = hoff[e];
        o.n_tracks = toff[e + 1] - toff[e]; o.n_track_hits = hoff[e + 1] - hoff[e];
        o.trk_sector = oi[0] + at; o.trk_first_hit = oi[1] + at; o.trk_n_hits = oi[2] + at; o.trk_ndf = oi[3] + at;
        o.trk_x = of[0] + at; o.trk_y = of[1] + at; o.trk_z = of[2] + at; o.trk_sinphi = of[3] + at; o.trk_tgl = of[4] + at;
        o.trk_qpt = of[5] + at; o.trk_chi2 = of[6] + at;
        o.hit_idx = ohit + ah;
        o.trk_out_x = rf ? of[7] + at : nullptr; o.trk_out_y = rf ? of[8] + at : nullptr; o.trk_out_z = rf ? of[9] + at : nullptr;
        o.trk_out_sinphi = rf ? of[10] + at : nullptr; o.trk_out_tgl = rf ? of[11] + at : nullptr;
        o.trk_out_qpt = rf ? of[12] + at : nullptr;
        o.trk_next = mg ? oi[4] + at : nullptr; o.trk_prev = mg ? oi[5] + at : nullptr; o.trk_global = mg ? oi[6] + at : nullptr;
        o.trk_g_ndf = mg ? oi[7] + at : nullptr; o.trk_g_n_hits = mg ? oi[8] + at : nullptr; o.trk_g_sector = mg ? oi[9] + at : nullptr;
        o.trk_g_x = mg ? of[13] + at : nullptr; o.trk_g_y = mg ? of[14] + at : nullptr; o.trk_g_z = mg ? of[15] + at : nullptr;
        o.trk_g_sinphi = mg ? of[16] + at : nullptr; o.trk_g_tgl = mg ? of[17] + at : nullptr; o.trk_g_qpt = mg ? of[18] + at : nullptr;
        o.trk_g_chi2 = mg ? of[19] + at : nullptr;
    }
    return TPC_OK;
}

int tpc_track_event(tpc_tracker* t, const tpc_event_in* in, tpc_event_out* out) { return tpc_track_events(t, 1, in, out); }

int tpc_tracker_set_profiling(tpc_tracker* t, int32_t on) {
    if (!t) return TPC_ERR_ARG;
    t->profiling = on != 0;
    return TPC_OK;
}

int tpc_get_stage_ms(const tpc_tracker* t, float* ms) {
    if (!t || !ms) return TPC_ERR_ARG;
    for (int k = 0; k < TPC_N_STAGES; k++) ms[k] = t->profiling ? t->stage_ms[k] : 0.f;
    return TPC_OK;
}

int tpc_get_counters(const tpc_tracker* t, tpc_counters* c) {
    if (!t || !c) return TPC_ERR_ARG;
    *c = t->counters;
    return TPC_OK;
}

// ---- intermediates (host-side conversion to the caller's indices; not on the hot path) ----
static int dbg_ranges(const tpc_tracker* tr, int& event, const Batch** bp, int* g0, int* g1, int* s0, int* s1) {
    if (!tr || !tr->have_result || event < 0 || event >= tr->n_events) { set_err("no result / bad event"); return TPC_ERR_ARG; }
    if (tr->ev_slot[event] < 0) { set_err("the intermediates of event %d have been overwritten by a later group", event); return TPC_ERR_ARG; }
    const Batch* t = tr->slots[tr->ev_slot[event]];
    event = tr->ev_local[event];
    *bp = t;
    const int bpe = tr->c.n_sectors * tr->c.n_rows;
    int32_t r[2], q[2];
    cudaStreamSynchronize(t->stream);
    if (cudaMemcpy(&r[0], t->v.bin_start + (size_t)event * bpe, 4, cudaMemcpyDeviceToHost) != cudaSuccess ||
        cudaMemcpy(&r[1], t->v.bin_start + (size_t)(event + 1) * bpe, 4, cudaMemcpyDeviceToHost) != cudaSuccess ||
        cudaMemcpy(&q[0], t->v.seed_start + (size_t)event * bpe, 4, cudaMemcpyDeviceToHost) != cudaSuccess ||
        cudaMemcpy(&q[1], t->v.seed_start + (size_t)(event + 1) * bpe, 4, cudaMemcpyDeviceToHost) != cudaSuccess) {
        set_err("cudaMemcpy failed in debug access");
        return TPC_ERR_CUDA;
    }
    *g0 = r[0]; *g1 = r[1]; *s0 = q[0]; *s1 = q[1];
    return TPC_OK;
}

int64_t tpc_debug_size(const tpc_tracker* tr, int32_t what, int32_t event) {
    int g0, g1, s0, s1;
    const Batch* t = nullptr;
    int rc = dbg_ranges(tr, event, &t, &g0, &g1, &s0, &s1);
    if (rc != TPC_OK) return rc;
    const int64_t n = g1 - g0, s = s1 - s0;
    switch (what) {
        case TPC_DBG_LINK_UP: case TPC_DBG_LINK_DN: case TPC_DBG_CLINK_UP: case TPC_DBG_CLINK_DN: case TPC_DBG_SORTED:
            return 4 * n;
        case TPC_DBG_START_HIT: return 4 * s;
        case TPC_DBG_TL_ROWS: return 12 * s;
        case TPC_DBG_TL_PAR: return 24 * s;
        case TPC_DBG_TL_TABLE: return 4 * s * tr->c.n_rows;
        default: set_err("unknown debug item"); return TPC_ERR_ARG;
    }
}

int tpc_debug_get(tpc_tracker* tr, int32_t what, int32_t event, void* buf, size_t bytes) {
    int g0, g1, s0, s1;
    const int64_t need = tpc_debug_size(tr, what, event);
    const Batch* t = nullptr;
    int rc = dbg_ranges(tr, event, &t, &g0, &g1, &s0, &s1);
    if (rc != TPC_OK) return rc;
    if (need < 0) return (int)need;
    if (!buf || bytes < (size_t)need) { set_err("debug buffer too small: need %lld bytes", (long long)need); return TPC_ERR_ARG; }
    const int n = g1 - g0, s = s1 - s0, nr = tr->c.n_rows;
    std::vector<int32_t> sorig(std::max(n, 1));
    if (n) CK(cudaMemcpy(sorig.data(), t->v.sorig + g0, 4 * (size_t)n, cudaMemcpyDeviceToHost));
    auto to_orig = [&](int32_t g) { return g < 0 ? -1 : sorig[g - g0]; };
    int32_t* ob = (int32_t*)buf;
    switch (what) {
        case TPC_DBG_SORTED: memcpy(buf, sorig.data(), 4 * (size_t)n); return TPC_OK;
        case TPC_DBG_LINK_UP: case TPC_DBG_LINK_DN: case TPC_DBG_CLINK_UP: case TPC_DBG_CLINK_DN: {
            const int32_t* src = what == TPC_DBG_LINK_UP ? t->v.link_up : what == TPC_DBG_LINK_DN ? t->v.link_dn
                                 : what == TPC_DBG_CLINK_UP ? t->v.clink_up : t->v.clink_dn;
            std::vector<int32_t> l(std::max(n, 1));
            if (n) CK(cudaMemcpy(l.data(), src + g0, 4 * (size_t)n, cudaMemcpyDeviceToHost));
            for (int k = 0; k < n; k++) ob[sorig[k]] = to_orig(l[k]);
            return TPC_OK;
        }
        case TPC_DBG_START_HIT: {
            std::vector<int32_t> l(std::max(s, 1));
            if (s) CK(cudaMemcpy(l.data(), t->v.seeds + s0, 4 * (size_t)s, cudaMemcpyDeviceToHost));
            for (int k = 0; k < s; k++) ob[k] = to_orig(l[k]);
            return TPC_OK;
        }
        case TPC_DBG_TL_ROWS: {
            std::vector<int32_t> l(std::max(s, 1));
            if (s) CK(cudaMemcpy(l.data(), t->v.tl_rows + s0, 4 * (size_t)s, cudaMemcpyDeviceToHost));
            for (int k = 0; k < s; k++) {
                const bool built = (l[k] >> 16) > 0;   // 0 hits: the start hit was skipped by the seed de-duplication
                ob[3 * k] = built ? (l[k] & 0xff) : -1; ob[3 * k + 1] = built ? ((l[k] >> 8) & 0xff) : -1; ob[3 * k + 2] = l[k] >> 16;
            }
            return TPC_OK;
        }
        case TPC_DBG_TL_PAR: {
            std::vector<float> l(std::max(s, 1));
            float* of = (float*)buf;
            for (int j = 0; j < 6; j++) {
                if (s) CK(cudaMemcpy(l.data(), t->v.tl_par + (size_t)j * t->S_cap + s0, 4 * (size_t)s, cudaMemcpyDeviceToHost));
                for (int k = 0; k < s; k++) of[6 * k + j] = l[k];
            }
            return TPC_OK;
        }
        case TPC_DBG_TL_TABLE: {
            if (!s) return TPC_OK;
            const int stride = t->v.tab_stride;
            std::vector<int32_t> rows(s), sbin(s);
            std::vector<uint16_t> tab((size_t)s * stride);
            const int bpe = tr->c.n_sectors * nr;
            std::vector<BinDesc> desc(bpe);
            CK(cudaMemcpy(rows.data(), t->v.tl_rows + s0, 4 * (size_t)s, cudaMemcpyDeviceToHost));
            CK(cudaMemcpy(sbin.data(), t->v.seed_bin + s0, 4 * (size_t)s, cudaMemcpyDeviceToHost));
            CK(cudaMemcpy(tab.data(), t->v.tl_tab + (size_t)s0 * stride, 2 * tab.size(), cudaMemcpyDeviceToHost));
            CK(cudaMemcpy(desc.data(), t->v.desc + (size_t)event * bpe, sizeof(BinDesc) * (size_t)bpe, cudaMemcpyDeviceToHost));
            for (int k = 0; k < s; k++) {
                const bool built = (rows[k] >> 16) > 0;
                const int first = built ? (rows[k] & 0xff) : 1, last = built ? ((rows[k] >> 8) & 0xff) : 0;
                const int tb = sbin[k] - sbin[k] % nr - event * bpe;   // first bin of the tracklet's task, event-local
                const uint16_t* tp = tab.data() + (size_t)k * stride;
                for (int r = 0; r < nr; r++)
                    ob[(size_t)k * nr + r] = (r >= first && r <= last && tp[r] != kNoHit) ? to_orig(desc[tb + r].base + tp[r]) : -1;
            }
            return TPC_OK;
        }
        default: set_err("unknown debug item"); return TPC_ERR_ARG;
    }
}

int tpc_measure_fp32_peak(float* fused_tflops, float* unfused_tflops) {
    if (!fused_tflops || !unfused_tflops) { set_err("null result pointers"); return TPC_ERR_ARG; }
    int dev = 0, sms = 0;
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const int blocks = sms * 8;                      // 2048 threads per SM: every scheduler has 16 warps to pick from
    float* d = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    float best[2] = {0.f, 0.f};
    cudaError_t e = cudaMalloc((void**)&d, 4);
    if (e == cudaSuccess) e = cudaEventCreate(&e0);
    if (e == cudaSuccess) e = cudaEventCreate(&e1);
    for (int fused = 0; fused < 2 && e == cudaSuccess; fused++)
        for (int rep = 0; rep < 6 && e == cudaSuccess; rep++) {   // first launches warm up; the best of the rest counts
            float ms = 0.f;
            e = cudaEventRecord(e0, 0);
            if (fused) k_fp32_peak<true><<<blocks, kPeakThreads>>>(d, 1.0000001f, 1.0e-7f);
            else k_fp32_peak<false><<<blocks, kPeakThreads>>>(d, 1.0000001f, 1.0e-7f);
            if (e == cudaSuccess) e = cudaEventRecord(e1, 0);
            if (e == cudaSuccess) e = cudaEventSynchronize(e1);
            if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
            if (e == cudaSuccess && rep >= 2 && ms > 0.f) best[fused] = std::max(best[fused], (float)(fp32_peak_flops_per_launch(blocks) / (ms * 1e-3) / 1e12));
        }
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e0) cudaEventDestroy(e0);      // the buffer and the events go on every path, failed or not
    if (e1) cudaEventDestroy(e1);
    if (d) cudaFree(d);
    if (e != cudaSuccess) { set_err("FP32 peak measurement failed: %s", cudaGetErrorString(e)); return TPC_ERR_CUDA; }
    *fused_tflops = best[1]; *unfused_tflops = best[0];
    return TPC_OK;
}

int tpc_debug_inject(tpc_tracker* tr, int32_t what, int32_t event, const void* buf, size_t bytes) {
    if (!tr || !tr->one_group) { set_err("inject needs a last call with device inputs that ran as one group"); return TPC_ERR_ARG; }
    const int64_t need = tpc_debug_size(tr, what, event);
    if (need < 0) return (int)need;
    int g0, g1, s0, s1;
    const Batch* tc = nullptr;
    int rc = dbg_ranges(tr, event, &tc, &g0, &g1, &s0, &s1);
    if (rc != TPC_OK) return rc;
    if (!buf || bytes != (size_t)need) { set_err("inject: the buffer must hold exactly %lld bytes", (long long)need); return TPC_ERR_ARG; }
    Batch* t = const_cast<Batch*>(tc);
    const int n = g1 - g0, s = s1 - s0, nr = tr->c.n_rows;
    std::vector<int32_t> sorig(std::max(n, 1)), inv(std::max(n, 1), -1);
    if (n) CK(cudaMemcpy(sorig.data(), t->v.sorig + g0, 4 * (size_t)n, cudaMemcpyDeviceToHost));
    for (int k = 0; k < n; k++) {
        if (sorig[k] < 0 || sorig[k] >= n) { set_err("inject: inconsistent work space"); return TPC_ERR_CUDA; }
        inv[sorig[k]] = g0 + k;   // caller's index -> sorted (batch-global) index
    }
    for (int i = 0; i < n; i++)   // the sorted order must name every cluster once, or inv[] has holes
        if (inv[i] < 0) { set_err("inject: the work space's sorted order is not a permutation of the event's clusters"); return TPC_ERR_CUDA; }
    const int32_t* ib = (const int32_t*)buf;
    switch (what) {
        case TPC_DBG_LINK_UP: case TPC_DBG_LINK_DN: case TPC_DBG_CLINK_UP: case TPC_DBG_CLINK_DN: {
            int32_t* dst = what == TPC_DBG_LINK_UP ? t->v.link_up : what == TPC_DBG_LINK_DN ? t->v.link_dn
                           : what == TPC_DBG_CLINK_UP ? t->v.clink_up : t->v.clink_dn;
            std::vector<int32_t> l(std::max(n, 1));
            for (int i = 0; i < n; i++) {
                const int32_t h = ib[i];
                if (h >= n) { set_err("inject: hit index %d outside the event", h); return TPC_ERR_ARG; }
                l[inv[i] - g0] = h < 0 ? -1 : inv[h];
            }
            if (n) CK(cudaMemcpy(dst + g0, l.data(), 4 * (size_t)n, cudaMemcpyHostToDevice));
            return TPC_OK;
        }
        case TPC_DBG_TL_ROWS: {
            std::vector<int32_t> l(std::max(s, 1));
            for (int k = 0; k < s; k++) {
                const int first = ib[3 * k], last = ib[3 * k + 1], nh = ib[3 * k + 2];
                if (nh < 0 || nh > nr || (nh > 0 && (first < 0 || last >= nr || first > last))) { set_err("inject: bad tracklet rows"); return TPC_ERR_ARG; }
                l[k] = nh > 0 ? (first | (last << 8) | (nh << 16)) : 0;
            }
            if (s) CK(cudaMemcpy(t->v.tl_rows + s0, l.data(), 4 * (size_t)s, cudaMemcpyHostToDevice));
            return TPC_OK;
        }
        case TPC_DBG_TL_PAR: {
            std::vector<float> l(std::max(s, 1));
            const float* fb = (const float*)buf;
            for (int j = 0; j < 6; j++) {
                for (int k = 0; k < s; k++) l[k] = fb[6 * k + j];
                if (s) CK(cudaMemcpy(t->v.tl_par + (size_t)j * t->S_cap + s0, l.data(), 4 * (size_t)s, cudaMemcpyHostToDevice));
            }
            return TPC_OK;
        }
        case TPC_DBG_TL_TABLE: {
            if (!s) return TPC_OK;
            const int stride = t->v.tab_stride;
            const int bpe = tr->c.n_sectors * nr;
            std::vector<int32_t> sbin(s);
            std::vector<uint16_t> tab((size_t)s * stride, kNoHit);
            std::vector<BinDesc> desc(bpe);
            CK(cudaMemcpy(sbin.data(), t->v.seed_bin + s0, 4 * (size_t)s, cudaMemcpyDeviceToHost));
            CK(cudaMemcpy(desc.data(), t->v.desc + (size_t)tr->ev_local[event] * bpe, sizeof(BinDesc) * (size_t)bpe, cudaMemcpyDeviceToHost));
            const int ev_bin0 = tr->ev_local[event] * bpe;
            for (int k = 0; k < s; k++) {
                const int tb = sbin[k] - sbin[k] % nr - ev_bin0;   // first bin of the tracklet's task, event-local
                for (int r = 0; r < nr; r++) {
                    const int32_t h = ib[(size_t)k * nr + r];
                    if (h < 0) continue;
                    if (h >= n) { set_err("inject: hit index %d outside the event", h); return TPC_ERR_ARG; }
                    const int loc = inv[h] - desc[tb + r].base;
                    if (loc < 0 || loc >= desc[tb + r].n) { set_err("inject: tracklet %d, row %d: the hit is not of that row", k, r); return TPC_ERR_ARG; }
                    tab[(size_t)k * stride + r] = (uint16_t)loc;
                }
            }
            CK(cudaMemcpy(t->v.tl_tab + (size_t)s0 * stride, tab.data(), 2 * tab.size(), cudaMemcpyHostToDevice));
            return TPC_OK;
        }
        default: set_err("this intermediate cannot be injected"); return TPC_ERR_ARG;
    }
}

int tpc_debug_resume(tpc_tracker* tr, int32_t from_stage, tpc_event_out* out) {
    if (!tr || !out || !tr->one_group) { set_err("resume needs a last call with device inputs that ran as one group"); return TPC_ERR_ARG; }
    if (from_stage < TPC_STAGE_CLEAN || from_stage > TPC_STAGE_SELECT) { set_err("resume: stage must be TPC_STAGE_CLEAN .. TPC_STAGE_SELECT"); return TPC_ERR_ARG; }
    Batch* t = tr->slots[0];
    const int n = t->n_events;
    cudaStream_t st = t->stream;
    CK(cudaStreamSynchronize(st));
    memset(&t->counters, 0, sizeof(tpc_counters));
    int rc = launch_all(tr, t, from_stage);
    if (rc != TPC_OK) return rc;
    CK(cudaMemcpyAsync(t->h_cnt.p, t->v.cnt, sizeof(unsigned long long) * CNT_N, cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(t->h_ev_off.p, t->v.ev_off, sizeof(int32_t) * 2 * (n + 1), cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(t->h_nseeds.p, t->v.seed_start + t->v.n_bins, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    const unsigned err = (unsigned)(t->h_cnt.p[CNT_ERR] & 0xffffffffu);
    if (err) { set_err("resume: the kernels reported error bits 0x%x (pools are not grown here)", err); return TPC_ERR_CAPACITY; }
    if (t->h_nseeds.p[0] > t->S_cap) { set_err("resume: more start hits than the tracklet pool holds"); return TPC_ERR_CAPACITY; }
    t->counters.n_events = n; t->counters.n_clusters = t->N;
    t->counters.n_links = (int64_t)t->h_cnt.p[CNT_LINKS]; t->counters.n_seeds = t->h_nseeds.p[0];
    t->counters.n_row_visits = (int64_t)t->h_cnt.p[CNT_ROW_VISITS]; t->counters.n_tracklet_hits = (int64_t)t->h_cnt.p[CNT_TL_HITS];
    t->counters.n_tracks = (int64_t)t->h_cnt.p[CNT_TRACKS]; t->counters.n_track_hits = (int64_t)t->h_cnt.p[CNT_TRACK_HITS];
    t->counters.n_updates = (int64_t)t->h_cnt.p[CNT_UPDATES]; t->counters.n_refit_visits = (int64_t)t->h_cnt.p[CNT_REFIT_VISITS];
    t->counters.n_tracklets = (int64_t)t->h_cnt.p[CNT_TRACKLETS];
    tr->counters = t->counters;
    const int32_t* toff = t->h_ev_off.p;
    const int32_t* hoff = t->h_ev_off.p + (n + 1);
    const bool rf = tr->c.p.refit != 0, mg = tr->c.p.merge != 0;
    for (int e = 0; e < n; e++) {
        tpc_event_out& o = out[e];
        const int64_t a = toff[e], h = hoff[e];
        o.n_tracks = toff[e + 1] - toff[e]; o.n_track_hits = hoff[e + 1] - hoff[e];
        o.trk_sector = t->o_i[0].p + a; o.trk_first_hit = t->o_i[1].p + a; o.trk_n_hits = t->o_i[2].p + a; o.trk_ndf = t->o_i[3].p + a;
        o.trk_x = t->o_f[0].p + a; o.trk_y = t->o_f[1].p + a; o.trk_z = t->o_f[2].p + a; o.trk_sinphi = t->o_f[3].p + a;
        o.trk_tgl = t->o_f[4].p + a; o.trk_qpt = t->o_f[5].p + a; o.trk_chi2 = t->o_f[6].p + a;
        o.hit_idx = t->v.o_hit_idx + h;
        o.trk_out_x = rf ? t->o_f[7].p + a : nullptr; o.trk_out_y = rf ? t->o_f[8].p + a : nullptr; o.trk_out_z = rf ? t->o_f[9].p + a : nullptr;
        o.trk_out_sinphi = rf ? t->o_f[10].p + a : nullptr; o.trk_out_tgl = rf ? t->o_f[11].p + a : nullptr;
        o.trk_out_qpt = rf ? t->o_f[12].p + a : nullptr;
        o.trk_next = mg ? t->o_i[4].p + a : nullptr; o.trk_prev = mg ? t->o_i[5].p + a : nullptr; o.trk_global = mg ? t->o_i[6].p + a : nullptr;
        o.trk_g_ndf = mg ? t->o_i[7].p + a : nullptr; o.trk_g_n_hits = mg ? t->o_i[8].p + a : nullptr; o.trk_g_sector = mg ? t->o_i[9].p + a : nullptr;
        o.trk_g_x = mg ? t->o_f[13].p + a : nullptr; o.trk_g_y = mg ? t->o_f[14].p + a : nullptr; o.trk_g_z = mg ? t->o_f[15].p + a : nullptr;
        o.trk_g_sinphi = mg ? t->o_f[16].p + a : nullptr; o.trk_g_tgl = mg ? t->o_f[17].p + a : nullptr; o.trk_g_qpt = mg ? t->o_f[18].p + a : nullptr;
        o.trk_g_chi2 = mg ? t->o_f[19].p + a : nullptr;
    }
    return TPC_OK;
}

// ---- prefix sum without any allocation (include/tpctrack.h "tpc_scan_exclusive_static") ----
//
// The tracker's prefix-sum kernel (scan.cuh: one launch, tiles that look back over their predecessors) needs a few
// words of global memory next to its input and output: a counter that hands out tile numbers and one status word per
// tile.  The tracker takes them from its cudaMalloc'ed work space.  The variant below takes them from an array that is
// part of the library image instead, so that a caller who must not (or cannot) allocate can still use the kernel.
//
// Size: one 8-byte word per tile of kScanTile = 2048 elements, plus the counter, for up to TPC_SCAN_STATIC_MAX_N
// elements = 8193 words, rounded up to 8 KiB words = 64 KiB + 256 B.  Every GPU that loads the library holds this much
// until the process exits.
namespace {
constexpr int kScanStaticWords = TPC_SCAN_STATIC_MAX_N / tpc::kScanTile + 1 + 31;
static_assert(TPC_SCAN_STATIC_MAX_N % tpc::kScanTile == 0, "the limit is a whole number of tiles");
static __device__ __align__(256) unsigned long long g_scan_static[kScanStaticWords];

// In host code `g_scan_static` is only a handle for the runtime (the host-side shadow of the device variable), NOT a
// device address: a kernel given `g_scan_static` or `&g_scan_static[0]` from the host would fault, or scribble over
// host memory on a system where the GPU can reach it.  The device address is asked for once per device, with that
// device current, and remembered here.
constexpr int kMaxDevices = 64;
unsigned long long* g_scan_static_addr[kMaxDevices] = {};
std::mutex g_scan_static_mutex;

int scan_static_address(unsigned long long** addr) {
    int dev = -1;
    CK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) { set_err("device ordinal %d is outside [0, %d)", dev, kMaxDevices); return TPC_ERR_ARG; }
    std::lock_guard<std::mutex> lock(g_scan_static_mutex);
    if (!g_scan_static_addr[dev]) {
        void* p = nullptr;
        CK(cudaGetSymbolAddress(&p, g_scan_static));   // the address on the CURRENT device (= dev)
        if (!p) { set_err("cudaGetSymbolAddress returned a null address on device %d", dev); return TPC_ERR_CUDA; }
        g_scan_static_addr[dev] = static_cast<unsigned long long*>(p);
    }
    *addr = g_scan_static_addr[dev];
    return TPC_OK;
}

int scan_check_args(const int32_t* in_dev, int64_t n, const int32_t* out_dev) {
    if (n < 0) { set_err("scan: n = %lld is negative", (long long)n); return TPC_ERR_ARG; }
    if (!out_dev || (n > 0 && !in_dev)) { set_err("scan: null device pointer"); return TPC_ERR_ARG; }
    return TPC_OK;
}
}  // namespace

int tpc_scan_exclusive_static(const int32_t* in_dev, int64_t n, int32_t* out_dev, void* cuda_stream) {
    int rc = scan_check_args(in_dev, n, out_dev);
    if (rc != TPC_OK) return rc;
    if (n > TPC_SCAN_STATIC_MAX_N) {
        set_err("tpc_scan_exclusive_static: n = %lld is beyond TPC_SCAN_STATIC_MAX_N = %d, the most the built-in scratch "
                "array serves (nothing was launched; cut the input or use a path that may allocate)",
                (long long)n, TPC_SCAN_STATIC_MAX_N);
        return TPC_ERR_CAPACITY;
    }
    unsigned long long* scratch = nullptr;
    rc = scan_static_address(&scratch);   // the first call on a device looks the address up; later calls read it back
    if (rc != TPC_OK) return rc;
    // The array still holds the tile counter and the status words of whoever used it last: scan_exclusive clears the
    // words this call will read (a memset on the same stream, in front of the kernel) -- nothing else must be zero.
    scan_exclusive(in_dev, out_dev, (int)n, scratch, static_cast<cudaStream_t>(cuda_stream));
    CK(cudaGetLastError());
    return TPC_OK;
}

int tpc_debug_scan_exclusive(const int32_t* in_dev, int64_t n, int32_t* out_dev) {
    int rc = scan_check_args(in_dev, n, out_dev);
    if (rc != TPC_OK) return rc;
    if (n > INT32_MAX - tpc::kScanTile) { set_err("scan: n = %lld is too large", (long long)n); return TPC_ERR_ARG; }
    unsigned long long* scratch = nullptr;
    CK(cudaMalloc((void**)&scratch, sizeof(unsigned long long) * ((size_t)n / tpc::kScanTile + 2)));
    scan_exclusive(in_dev, out_dev, (int)n, scratch, nullptr);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaStreamSynchronize(nullptr);
    cudaFree(scratch);
    if (e != cudaSuccess) { set_err("scan failed: %s", cudaGetErrorString(e)); return TPC_ERR_CUDA; }
    return TPC_OK;
}

}  // extern "C"
