/*
 * tpctrack.h -- C ABI of libtpctrack.so: the data-parallel hot path of the ALICE HLT TPC sector tracker
 * (arxiv 1712.09416) on one NVIDIA B200 (sm_100a).
 *
 * What it computes.  "our TPC tracker ... bases on a Cellular Automaton and on the Kalman filter"
 * (abstract; section 2).  The paper names no further step; the step list is the
 * contract of BASELINE.json:5: per-row cluster sort + uniform (y,z) grid; Cellular-Automaton neighbour finding
 * between adjacent pad rows (best up/down pair by straight-line deviation); mutual-link cleaning; start-hit
 * selection; Kalman-filter tracklet construction (float32 helix fit, state y, z, sin phi, tg lambda, q/pT in
 * sector-local coordinates); tracklet selection resolving shared hits.  The entry points are the ones that
 * sentence lists: tpc_tracker_create(geometry, Bz), tpc_track_event(clusters as SoA x,y,z,row -> tracks with hit
 * lists and helix parameters), tpc_tracker_destroy; plus the batch form for "several events concurrently".
 * The exact arithmetic of every step is written out in DESIGN.md ("The method, step by step").
 *
 * Every step runs in hand-written CUDA kernels; there is no CPU fallback.  Plain C types only.
 * A tracker is not thread-safe: one per host thread.  No exception crosses this boundary.
 */
#ifndef TPCTRACK_H
#define TPCTRACK_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* ---- status codes (0 = ok, negative = error) ---- */
#define TPC_OK 0
#define TPC_ERR_ARG (-1)       /* NULL pointer, bad size, row outside [0,n_rows), non-monotonic sector_offset */
#define TPC_ERR_GEOMETRY (-2)  /* row_x not strictly increasing, n_rows not in [3,255], n_sectors < 1 */
#define TPC_ERR_CAPACITY (-3)  /* more than TPC_MAX_ROW_HITS clusters in one (sector,row), or a pool limit */
#define TPC_ERR_CUDA (-4)      /* a CUDA call failed; tpc_last_error() has the text */

#define TPC_MAX_ROWS 255
#define TPC_MAX_ROW_HITS 2048  /* clusters per (sector, pad row); a fuller row makes the call fail with TPC_ERR_CAPACITY
                                * (row-local hit numbers are 16-bit and the row sort works in shared memory) */

/* Geometry of the detector (copied at create; host pointers).  Units: cm, Tesla, GeV/c.
 * Sector-local frame: x along the sector axis (a cluster of pad row r sits at x = row_x[r] exactly), y across,
 * z along the drift (signed: C-side sectors have z < 0).  BASELINE.json:7: 159 rows, 20 degree wedges. */
typedef struct {
    int32_t n_sectors;         /* 36 (or 1): the number of independent sector tasks per event; 1..64 (more is
                                * TPC_ERR_GEOMETRY: the first kernels keep an event's sector offsets in shared memory) */
    int32_t n_rows;            /* pad rows per sector, 3..TPC_MAX_ROWS */
    const float* row_x;        /* [n_rows] host, strictly increasing */
    float tan_half_angle;      /* tan(10 deg): the wedge is |y| <= row_x * tan_half_angle */
    float z_abs_max;           /* 250 cm, informational */
    float sigma_y, sigma_z;    /* cluster errors used by the fit, cm */
    const float* sector_alpha; /* [n_sectors] host or NULL; echoed only, tracking is sector-local */
} tpc_geometry;

/* Algorithm parameters (defaults from tpc_default_params). */
typedef struct {
    int32_t link_step;          /* Delta: neighbour rows r +- Delta, 1 or 2 */
    float nf_slope_y, nf_slope_z; /* neighbour window half width = slope * |dx| + nf_w0 */
    float nf_w0;                /* cm */
    float nf_dmax;              /* largest accepted straight-line deviation, cm^2 */
    float sin_max;              /* the helix transport fails beyond |sin phi| = sin_max */
    float var_s, var_t, var_q;  /* prior variances of sin phi, tg lambda, q/pT */
    float chi2_link, chi2_ext;  /* 2-dof gates: following a link / attaching a searched hit */
    float win_nsigma, win_min, win_max; /* search window = clamp(n * sqrt(C + sigma^2), min, max) cm */
    int32_t max_gap;            /* consecutive rows without a hit before a pass ends, 0..60 */
    float edge_margin;          /* cm beyond the wedge edge before a pass ends */
    int32_t min_tracklet_hits;  /* tracklets with fewer hits do not take part in the selection */
    int32_t min_track_hits;     /* tracks keeping fewer owned hits are dropped */
    int32_t refit;              /* 0 (default): track parameters are the tracklet's (no refit).  1: every output
                                 * track is refitted over its final hit list: up
                                 * pass from its lowest hit, fresh down pass from the top hit reached, no search, no
                                 * gate; trk_x/y/z/sinphi/tgl/qpt/chi2/ndf are then the refit's (x = row of the
                                 * lowest hit the down pass reached, ndf = 2 * hits in the refit - 5) */
    int32_t merge;              /* 1: link the track segments of one particle across sector borders (O9, SURVEY.md
                                 * 8(f).2; needs refit = 1): trk_next / trk_prev / trk_global, and fit every global
                                 * track over all its segments (O10): trk_g_*.  Sectors: n_sectors / 2 per side,
                                 * sector s = side * (n_sectors / 2) + k at azimuth (k + 1/2) * 4 pi / n_sectors */
    float merge_dy, merge_dz;   /* cm: tolerated |dy|, |dz| between the extrapolated and the found segment */
    float merge_ds, merge_dt;   /* tolerated |d sin phi|, |d tg lambda| */
    int32_t merge_max_gap;      /* pad rows that may be missing between the two segments */
    int32_t seed_dedup;         /* 1 (default): a start hit that the up pass of a tracklet built from a lower pad row of
                                 * its sector has already recorded builds no tracklet (R23).
                                 * 0: every start hit is fitted (round-1 behaviour, ~3 tracklets per output track) */
    int32_t checked;            /* 0 (default) fast mode: cluster coordinates are trusted; a non-finite y or z, or an x
                                 * that is not row_x[row], gives undefined TRACKS (never a memory fault; a row outside
                                 * [0, n_rows) is still reported).  1 checked mode: the first
                                 * kernel also tests every cluster -- y, z finite, and, where x is given (non-NULL),
                                 * |x - row_x[row]| <= 1e-3 cm -- and the call returns TPC_ERR_ARG otherwise */
} tpc_params;

/* One event's clusters: SoA, grouped by sector, ANY order inside a sector.  Fast mode (tpc_params.checked = 0) trusts
 * the coordinates: see tpc_params.checked.
 * mem_space 0: x, y, z, row are host pointers; the call copies them to the device (pinned memory makes the
 *              copy asynchronous) and the outputs come back in library-owned pinned host memory.
 * mem_space 1: x, y, z, row are device pointers (must stay valid and unchanged until the call returns); the
 *              outputs are library-owned device memory.
 * sector_offset is ALWAYS a host pointer.  x is redundant with row_x[row]: the library reads row and ignores x
 * (x may be NULL), except in checked mode, which compares the two. */
typedef struct {
    int32_t n_clusters;
    const int32_t* sector_offset; /* [n_sectors+1] host, non-decreasing, [0] = 0, [n_sectors] = n_clusters */
    const float* x;
    const float* y;
    const float* z;
    const int32_t* row;           /* [n_clusters] in [0, n_rows) */
    int32_t mem_space;
} tpc_event_in;

/* One event's tracks.  All arrays are library-owned (host or device as the input's mem_space) and valid until
 * the next tpc_track_event(s) call on this tracker or its destruction.  Tracks come in canonical order
 * (sector, pad row of the start hit, caller's index of the start hit).  A hit is in at most one track.
 * Parameters are given at x = trk_x (the pad row of the track's innermost fitted hit). */
typedef struct {
    int32_t n_tracks;
    int32_t n_track_hits;
    const int32_t* trk_sector;    /* [n_tracks] */
    const int32_t* trk_first_hit; /* [n_tracks] offset into hit_idx */
    const int32_t* trk_n_hits;    /* [n_tracks] hits this track owns */
    const int32_t* trk_ndf;       /* [n_tracks] 2 * (hits in the fit) - 5 */
    const float* trk_x;           /* [n_tracks] cm */
    const float* trk_y;
    const float* trk_z;
    const float* trk_sinphi;
    const float* trk_tgl;
    const float* trk_qpt;         /* 1/(GeV/c), signed */
    const float* trk_chi2;
    const int32_t* hit_idx;       /* [n_track_hits] indices into the caller's cluster arrays, row-ascending */
    /* tpc_params.refit = 1 (NULL otherwise): the refit's OUTER state, i.e. its up pass right after the update with
     * the track's top hit, at x = trk_out_x (all hits of the track are in it; it is what extrapolates outwards) */
    const float* trk_out_x;       /* [n_tracks] cm */
    const float* trk_out_y;
    const float* trk_out_z;
    const float* trk_out_sinphi;
    const float* trk_out_tgl;
    const float* trk_out_qpt;
    /* tpc_params.merge = 1 (NULL otherwise): the segment that continues this one in a neighbouring sector /
     * the segment this one continues; index into this event's tracks or -1.  Links are mutual and one-to-one. */
    const int32_t* trk_next;      /* [n_tracks] */
    const int32_t* trk_prev;      /* [n_tracks] */
    const int32_t* trk_global;    /* [n_tracks] the global track a segment belongs to = the chain of linked segments,
                                   * named by the index of its first (innermost) segment */
    /* tpc_params.merge = 1: the fit of the global track over the hits of ALL its segments (up and
     * down pass as the refit, the fit turned into the next sector's frame at each border), stored at the chain's
     * first segment i = trk_global[...]: parameters at x = trk_g_x[i] in the frame of sector trk_g_sector[i]
     * (normally the first segment's).  A lone segment's global fit is its refit; entries of segments that are not
     * the first of their chain are 0 (trk_g_sector -1). */
    const float* trk_g_x;         /* [n_tracks] cm */
    const float* trk_g_y;
    const float* trk_g_z;
    const float* trk_g_sinphi;
    const float* trk_g_tgl;
    const float* trk_g_qpt;
    const float* trk_g_chi2;
    const int32_t* trk_g_ndf;     /* [n_tracks] 2 * trk_g_n_hits - 5 */
    const int32_t* trk_g_n_hits;  /* [n_tracks] hits in the global fit */
    const int32_t* trk_g_sector;  /* [n_tracks] */
} tpc_event_out;

/* Counters of the last call (whole batch); used for the algorithmic-byte count of DESIGN.md. */
typedef struct {
    int64_t n_events, n_clusters;
    int64_t n_links;         /* hits with a cleaned up-link */
    int64_t n_seeds;         /* start hits (with seed_dedup only part of them build a tracklet: n_tracklets) */
    int64_t n_row_visits;    /* Kalman transport steps taken by the constructor */
    int64_t n_tracklet_hits; /* hits in tracklets entering the selection */
    int64_t n_tracks, n_track_hits;
    int64_t n_kernel_launches; /* kernels this library launched during the call */
    int64_t n_retries;       /* internal re-runs after growing a pool */
    int64_t n_updates;       /* Kalman updates (accepted measurements, both passes) */
    int64_t n_refit_visits;  /* row visits of the refit (0 when tpc_params.refit is 0) */
    int64_t n_tracklets;     /* tracklets constructed (start hits not skipped by the seed de-duplication) */
} tpc_counters;

typedef struct tpc_tracker tpc_tracker;

/* Fill *p with the defaults. */
void tpc_default_params(tpc_params* p);

/* Create a tracker for the given geometry and solenoid field Bz (Tesla, signed).  Default parameters; work
 * space grows on demand.  Returns NULL on failure (tpc_last_error()). */
tpc_tracker* tpc_tracker_create(const tpc_geometry* geometry, float bz_tesla);

/* As above with explicit parameters (NULL = defaults) and pre-sized work space: the tracker allocates once
 * for batches of up to max_events events holding up to max_clusters clusters in total (0 = grow on demand). */
tpc_tracker* tpc_tracker_create_ex(const tpc_geometry* geometry, float bz_tesla, const tpc_params* params,
                                   int32_t max_events, int64_t max_clusters);

/* Run all kernels on this CUDA stream (a cudaStream_t; NULL = the tracker's own stream). */
int tpc_tracker_set_stream(tpc_tracker* t, void* cuda_stream);

/* Host-input batches (mem_space 0) are cut into groups of events that run on separate streams, so that the copies
 * of one group overlap the kernels of another ("several events ... processed concurrently on one GPU via streams",
 * BASELINE.json:5).  n = events per group; 0 (default) = automatic (up to four groups of at least ~2 M clusters).
 * Results do not depend on the grouping.  Device-input batches run as one group unless n > 0 is set, in which
 * case they are cut into at most four groups whose kernels may overlap on the device. */
int tpc_tracker_set_group_events(tpc_tracker* t, int32_t n);

/* Track one event.  Synchronous: returns when the outputs are complete.  Zero clusters, empty sectors and
 * empty rows are legal (0 tracks).  Returns a status code. */
int tpc_track_event(tpc_tracker* t, const tpc_event_in* in, tpc_event_out* out);

/* Track n independent events in one pass: all n * n_sectors sector tasks go through every kernel together.
 * in/out are host arrays of n structs; all inputs must share one mem_space. */
int tpc_track_events(tpc_tracker* t, int32_t n, const tpc_event_in* in, tpc_event_out* out);

/* The same pass in two halves, so that up to three batches can be in flight: while the kernels of one batch run, the
 * clusters of the next are copied in and the tracks of the one before are copied out ("asynchronous data
 * processing", the paper's title; the sync call above exposes those copies).
 * tpc_submit_events enqueues the input copies and all kernels of a batch on a stream of its own and returns at once
 * with a ticket (0, 1 or 2); at most three batches are in flight (a fourth submit returns TPC_ERR_ARG).  The `in` array,
 * the sector offsets and the cluster arrays must stay valid and unchanged until the matching wait returns.
 * tpc_wait_events waits for that batch, copies the outputs back (host inputs) and fills out[0..n).  The outputs
 * are library-owned (each ticket has its own output arrays, host or device) and stay valid until the next wait on
 * the same ticket number -- so at least until the second submit after this wait -- or destroy.  The batch runs as one
 * group; results are those of tpc_track_events.  Intermediates (tpc_debug_get) are not kept for these batches. */
int tpc_submit_events(tpc_tracker* t, int32_t n, const tpc_event_in* in, int32_t* ticket);
int tpc_wait_events(tpc_tracker* t, int32_t ticket, tpc_event_out* out);

void tpc_tracker_destroy(tpc_tracker* t);

const char* tpc_status_string(int status);
const char* tpc_last_error(void); /* thread-local text of the last failure */

int tpc_get_counters(const tpc_tracker* t, tpc_counters* c);

/* Per-stage device times of the last call, measured with CUDA events on the tracker's stream (off by default:
 * the events cost a few microseconds).  Stages: 0 = K1 bucket + grid sort, 1 = K2 neighbour finder,
 * 2 = K3 cleaner + K4 start hits, 3 = K5 tracklet constructor (one launch: up and down sweep of every sector task),
 * 4 = K6 selector + output, 5 = refit of the output tracks (0 when tpc_params.refit is 0). */
#define TPC_N_STAGES 6
int tpc_tracker_set_profiling(tpc_tracker* t, int32_t on);
int tpc_get_stage_ms(const tpc_tracker* t, float* ms /* [TPC_N_STAGES] */);

/* Measured FP32 arithmetic peaks of the current device, in TFLOP/s (multiply and add counted separately): independent
 * chains of fused multiply-adds, and of un-fused multiply + add pairs -- the ceiling of arithmetic that is defined
 * without contraction, as this tracker's is.  The denominators of the constructor's
 * roofline in bench.py; takes a few milliseconds; not part of the hot path. */
int tpc_measure_fp32_peak(float* fused_tflops, float* unfused_tflops);

/* ---- intermediates of the last call, for stage-by-stage parity tests (not part of the hot path) ----
 * All hit indices are the caller's indices within event `event`; -1 = none.  buf is a HOST buffer of `bytes`
 * bytes; the call fails with TPC_ERR_ARG if it is too small.  Sizes: tpc_debug_size().  After a host-input batch
 * that ran as more than three groups only the events of the last three groups still have their intermediates
 * (TPC_ERR_ARG for the others). */
#define TPC_DBG_LINK_UP 0    /* int32 [n_clusters(event)]  neighbour before cleaning */
#define TPC_DBG_LINK_DN 1
#define TPC_DBG_CLINK_UP 2   /* int32 [n_clusters(event)]  after cleaning */
#define TPC_DBG_CLINK_DN 3
#define TPC_DBG_START_HIT 4  /* int32 [n_seeds(event)]     canonical order */
#define TPC_DBG_TL_ROWS 5    /* int32 [n_seeds(event)][3]  first_row, last_row, n_hits */
#define TPC_DBG_TL_PAR 6     /* float [n_seeds(event)][6]  y, z, sin phi, tg lambda, q/pT, chi2 */
#define TPC_DBG_TL_TABLE 7   /* int32 [n_seeds(event)][n_rows] row -> hit */
#define TPC_DBG_SORTED 8     /* int32 [n_clusters(event)]  caller's index of each cluster in (sector,row,cell) order */
int64_t tpc_debug_size(const tpc_tracker* t, int32_t what, int32_t event); /* bytes, or negative status */
int tpc_debug_get(tpc_tracker* t, int32_t what, int32_t event, void* buf, size_t bytes);

/* ---- stage-isolated parity ("GPU stage k on the reference's output of stage k-1") ----
 * tpc_debug_inject overwrites one intermediate of event `event` of the last call with the caller's values (same
 * layouts, sizes and index convention as tpc_debug_get; buf is a HOST buffer of exactly tpc_debug_size bytes).
 * Items: TPC_DBG_LINK_UP / LINK_DN (input of K3), TPC_DBG_CLINK_UP / CLINK_DN (input of K4 and K5),
 * TPC_DBG_TL_ROWS / TL_PAR / TL_TABLE (input of K6; rows with n_hits = 0 mean "no tracklet").  The start-hit list
 * is not injectable: it is a function of the cleaned links (K4).
 * tpc_debug_resume then runs the path again FROM a stage on what the work space now holds, for all events of
 * the last call, and fills out[0 .. n_events) like the call itself did:
 *   TPC_STAGE_CLEAN (K3, K4, K5, K6): after injecting links;
 *   TPC_STAGE_SEEDS (K4 from the cleaned links as they stand, K5, K6): after injecting cleaned links;
 *   TPC_STAGE_CONSTRUCT (K5, K6);  TPC_STAGE_SELECT (K6 only): after injecting tracklets.
 * Both need a last call with device inputs (mem_space 1) made through tpc_track_event(s) that ran as one group, and
 * return TPC_ERR_ARG otherwise.  The counters afterwards cover the stages that ran again. */
#define TPC_STAGE_CLEAN 3
#define TPC_STAGE_SEEDS 4
#define TPC_STAGE_CONSTRUCT 5
#define TPC_STAGE_SELECT 6
int tpc_debug_inject(tpc_tracker* t, int32_t what, int32_t event, const void* buf, size_t bytes);
int tpc_debug_resume(tpc_tracker* t, int32_t from_stage, tpc_event_out* out);

/* ---- a prefix sum for callers that cannot allocate device memory ----
 * Who this is for.  The tracker sizes its work space with cudaMalloc (at create, and again when a batch outgrows a
 * pool).  Some users of its kernels have no such freedom: an online reconstruction process in which a framework
 * reserved the whole GPU memory at start-up and forbids its components to ask the driver for more (a cudaMalloc there
 * fails, or breaks the framework's accounting); code on a path with a latency bound, where cudaMalloc and cudaFree
 * are ruled out because they may stall every stream of the device for an unbounded time; a plug-in that is only handed
 * input and output buffers.  For them the library carries ONE entry point that never allocates: the tracker's
 * exclusive prefix sum of int32 (the step between "count per (sector, pad row) bin" and "offset of each bin" in K1, K4
 * and K6; BASELINE.json:5 "per-row cluster sort"), with the few words of scratch memory the kernel needs (a tile
 * counter and one status word per tile of 2048 elements) taken from an array that is part of the library image.
 *
 *   out_dev[i] = in_dev[0] + ... + in_dev[i-1]  for i = 0 .. n   (out_dev[0] = 0, out_dev[n] = the total; int32
 *   arithmetic, wraps on overflow like the tracker's own).  in_dev [n] and out_dev [n + 1] are DEVICE pointers owned by
 *   the caller, 4-byte aligned, not overlapping; in_dev may be NULL when n = 0.
 *
 * Limit.  n <= TPC_SCAN_STATIC_MAX_N (16 Mi elements; the array is 64 KiB + 256 B, held by every GPU that loads the
 * library until the process ends).  A larger n returns TPC_ERR_CAPACITY with the reason in tpc_last_error() and
 * launches nothing; n < 0 or a NULL pointer returns TPC_ERR_ARG.
 * No allocation.  The call makes no cudaMalloc, cudaFree, cudaMallocHost or any library call that allocates: it
 * enqueues one memset of the scratch words it is about to use and one kernel on `cuda_stream` (a cudaStream_t; NULL =
 * the default stream) and returns without waiting; the result is complete when that stream has run them.
 * First call on a device.  It looks up where the built-in array lives on the current device (cudaGetSymbolAddress,
 * once per device, kept for later calls; this may make the CUDA runtime load the library's device code).  Make this
 * first call during set-up, with the device that will be used current, and before any stream capture is begun.
 * One array for everybody.  All calls on a device -- from any thread, stream or tracker -- share that array, and it
 * keeps what the previous call left in it.  The call clears the words it needs itself, so calls that follow one
 * another on one stream (or are ordered by events) are independent; two calls whose kernels can overlap on the GPU
 * race on the array and give wrong sums -- the caller must keep them apart. */
#define TPC_SCAN_STATIC_MAX_N (1 << 24)
int tpc_scan_exclusive_static(const int32_t* in_dev, int64_t n, int32_t* out_dev, void* cuda_stream);

/* The same prefix sum the way the tracker itself runs it, for tests: same kernel, scratch words from cudaMalloc, freed
 * before the call returns; default stream, synchronous.  n up to 2^31 - 2049.  Not for the hot path. */
int tpc_debug_scan_exclusive(const int32_t* in_dev, int64_t n, int32_t* out_dev);

#ifdef __cplusplus
}
#endif
#endif /* TPCTRACK_H */
