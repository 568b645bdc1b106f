"""The constructor's (K5) other state-slot tiers under parity (-m gpu, through the C ABI).

K5 keeps the state of every tracklet under way in a slot: tier 0 = 512 shared-memory slots and two CTAs per SM (batches
with more sector tasks than SMs), tier 1 = 1408 slots and one CTA per SM (single events), tier 2 = 1280 shared-memory
+ 4096 GLOBAL-memory slots per CTA.  A launch that runs out of slots reports it, and the host runs the batch again one
tier higher and stays there (csrc/tracker.cu `batch_finish`).  The parity tests of test_gpu_parity.py reach tiers 0 and
1 only; here the tier is forced with TPCTRACK_CT_TIER (read when a tracker is created) and the run-time move is
provoked with seed_dedup = 0, which triples the tracklets under way (R23).

Every result is compared with the oracle's strict-float32 mode: integers exactly, parameters within 1e-4
(SURVEY.md 8(c).6)."""
import numpy as np
import pytest

from conftest import make_geometry
from test_gpu_parity import TOL, compare_event, copy_params, ev_dict, make_tracker, trk_mod  # noqa: F401

pytestmark = pytest.mark.gpu

_refs = {}


def oracle_of(oracle_mod, gen_mod, name, event, dedup):
    key = (name, event, dedup)
    if key not in _refs:
        ev = gen_mod.generate(name, event)
        p = oracle_mod.default_params()
        p.seed_dedup = dedup
        _refs[key] = (ev, oracle_mod.track_event(make_geometry(oracle_mod, gen_mod, ev), ev.sector_offset, ev.y, ev.z,
                                                 ev.row, params=p, precision="float"))
    return _refs[key]


def params_of(oracle_mod, trk_mod, dedup):
    p = oracle_mod.default_params()
    p.seed_dedup = dedup
    return copy_params(p, trk_mod)


def tracks_equal(res, ref, what):
    assert res["n_tracks"] == ref.n_tracks and res["n_track_hits"] == ref.n_track_hits, what
    for k in ("trk_sector", "trk_first_hit", "trk_n_hits", "trk_ndf", "hit_idx"):
        assert np.array_equal(res[k], ref[k]), (what, k)
    for k in ("trk_x", "trk_y", "trk_z", "trk_sinphi", "trk_tgl", "trk_qpt", "trk_chi2"):
        err = np.abs(res[k] - ref[k]) / np.maximum(1.0, np.abs(ref[k]))
        assert err.max(initial=0.0) <= TOL, (what, k, err.max())


@pytest.mark.parametrize("name,dedup", [("single_sector", 1), ("semicentral", 1), ("semicentral", 0), ("central", 0)])
def test_parity_in_tier_2(trk_mod, gen_mod, oracle_mod, monkeypatch, name, dedup):
    """TPCTRACK_CT_TIER=2: `k_construct<20, true, 1280>`, the variant whose slots beyond the first 1280 live in global
    memory.  Every stage's output compared.  The central event without seed de-duplication has more than 1408
    tracklets under way in a sector task (it does not fit tier 1: see the escalation test), so its fits do run in
    global-memory slots."""
    monkeypatch.setenv("TPCTRACK_CT_TIER", "2")
    ev, ref = oracle_of(oracle_mod, gen_mod, name, 0, dedup)
    trk = make_tracker(trk_mod, gen_mod, ev, params=params_of(oracle_mod, trk_mod, dedup))
    out = trk.tpc_track_event(ev_dict(ev, True))
    flips, _ = compare_event(trk, out, ev, ref)
    assert flips == 0
    assert trk.tpc_get_counters()["n_retries"] == 0
    trk.close()


def test_tier_moves_up_at_run_time_and_stays(trk_mod, gen_mod, oracle_mod, monkeypatch):
    """Five central events = 180 sector tasks (more than SMs), forced to START in tier 0 although every start hit is
    fitted: the tasks run out of the 512 slots, the launch reports kErrSlotCapacity, and tpc_track_events runs the batch
    again in the next tier -- twice, because 1408 slots are not enough either, so the batch ends in tier 2 with one CTA
    per SM serving more tasks than there are SMs.  Results are the oracle's; the second call starts in the tier the
    first one ended in."""
    monkeypatch.setenv("TPCTRACK_CT_TIER", "0")
    pairs = [oracle_of(oracle_mod, gen_mod, "central", e, 0) for e in range(5)]
    evs = [ev for ev, _ in pairs]
    trk = make_tracker(trk_mod, gen_mod, evs[0], params=params_of(oracle_mod, trk_mod, 0))
    outs = trk.tpc_track_events([ev_dict(ev, True) for ev in evs])
    c = trk.tpc_get_counters()
    assert c["n_retries"] == 2, c                                                      # tier 0 -> 1 -> 2
    assert c["n_tracklets"] == c["n_seeds"] == sum(ref.n_seeds for _, ref in pairs)   # counters are the last run's only
    for e, (ev, ref) in enumerate(pairs):
        flips, _ = compare_event(trk, outs[e], ev, ref, event=e)
        assert flips == 0
    outs = trk.tpc_track_events([ev_dict(ev, True) for ev in evs])
    assert trk.tpc_get_counters()["n_retries"] == 0                                     # the tier is sticky
    for e, (ev, ref) in enumerate(pairs):
        tracks_equal(trk.to_numpy(outs[e]), ref, e)
    trk.close()


def test_tier_2_groups_on_their_own_streams_keep_their_slots_apart(trk_mod, gen_mod, oracle_mod, monkeypatch):
    """Four central events as four groups on four streams, all in tier 2 with every start hit fitted: the four K5
    launches (36 CTAs each) can be resident together, and CTAs with equal blockIdx.x of different launches must not
    share global-memory slots (each group has its own slot array; one array per tracker once corrupted tracklets
    here)."""
    monkeypatch.setenv("TPCTRACK_CT_TIER", "2")
    pairs = [oracle_of(oracle_mod, gen_mod, "central", e, 0) for e in range(4)]
    evs = [ev for ev, _ in pairs]
    trk = make_tracker(trk_mod, gen_mod, evs[0], params=params_of(oracle_mod, trk_mod, 0))
    trk.tpc_tracker_set_group_events(1)
    for rep in range(3):
        outs = trk.tpc_track_events([ev_dict(ev, True) for ev in evs])
        for e, (ev, ref) in enumerate(pairs):
            tracks_equal(trk.to_numpy(outs[e]), ref, (rep, e))
    trk.close()


def test_tier_2_tickets_in_flight_keep_their_slots_apart(trk_mod, gen_mod, oracle_mod, monkeypatch):
    """The same through tpc_submit_events / tpc_wait_events: three batches in flight, each on its own stream."""
    monkeypatch.setenv("TPCTRACK_CT_TIER", "2")
    pairs = [oracle_of(oracle_mod, gen_mod, "central", e, 0) for e in range(3)]
    trk = make_tracker(trk_mod, gen_mod, pairs[0][0], params=params_of(oracle_mod, trk_mod, 0))
    d = [[ev_dict(ev, True)] for ev, _ in pairs]
    for rep in range(2):
        tickets = [trk.tpc_submit_events(x) for x in d]
        for e, tk in enumerate(tickets):
            tracks_equal(trk.to_numpy(trk.tpc_wait_events(tk)[0]), pairs[e][1], (rep, e))
    trk.close()
