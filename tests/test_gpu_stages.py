"""Stage-isolated GPU parity ("GPU stage k on the reference's output of stage k-1", through
tpc_debug_inject / tpc_debug_resume), the checked mode (S23), and the boundary's corner cases the round-1 review
found (-m gpu, through the C ABI).

Stage isolation is made non-trivial by injecting the intermediates of an oracle run with DIFFERENT parameters in
the stages BEFORE the one under test (the stage under test and everything after it run with the tracker's own
parameters on both sides): had the GPU stage ignored the injection and used its own upstream results, the
comparison would fail.
"""
import numpy as np
import pytest

from conftest import make_geometry
from test_gpu_parity import TOL, compare_event, copy_params, ev_dict, make_tracker, trk_mod  # noqa: F401

pytestmark = pytest.mark.gpu


def _oracle(oracle_mod, gen_mod, ev, **kw):
    p = oracle_mod.default_params()
    for k, v in kw.items():
        setattr(p, k, v)
    return oracle_mod.track_event(make_geometry(oracle_mod, gen_mod, ev), ev.sector_offset, ev.y, ev.z, ev.row, params=p,
                                  precision="float")


def _tracks_equal(res, ref):
    assert res["n_tracks"] == ref.n_tracks and res["n_track_hits"] == ref.n_track_hits
    for k in ("trk_sector", "trk_first_hit", "trk_n_hits", "trk_ndf", "hit_idx"):
        assert np.array_equal(res[k], ref[k]), k
    for k in ("trk_x", "trk_y", "trk_z", "trk_sinphi", "trk_tgl", "trk_qpt", "trk_chi2"):
        err = np.abs(res[k] - ref[k]) / np.maximum(1.0, np.abs(ref[k]))
        assert err.max(initial=0.0) <= TOL, (k, err.max())


@pytest.mark.parametrize("name", ["single_sector", "semicentral"])
def test_k3_k4_on_the_oracles_links(trk_mod, gen_mod, oracle_mod, name):
    """K3 + K4 (and everything after) on the links of an oracle run whose neighbour finder had other cuts."""
    ev = gen_mod.generate(name)
    other = _oracle(oracle_mod, gen_mod, ev, nf_dmax=0.05, nf_w0=0.2)       # O2 differs; O3.. identical
    own = _oracle(oracle_mod, gen_mod, ev)
    assert not np.array_equal(other.link_up, own.link_up)
    trk = make_tracker(trk_mod, gen_mod, ev)
    trk.tpc_track_event(ev_dict(ev, True))
    trk.tpc_debug_inject("link_up", other.link_up)
    trk.tpc_debug_inject("link_dn", other.link_dn)
    out = trk.tpc_debug_resume("clean")[0]
    for k in ("link_up", "link_dn", "clink_up", "clink_dn", "start_hit"):
        assert np.array_equal(trk.tpc_debug_get(k), other[k]), k
    assert np.array_equal(trk.tpc_debug_get("tl_table"), other.tl_table)
    _tracks_equal(trk.to_numpy(out), other)
    c = trk.tpc_get_counters()
    assert c["n_seeds"] == other.n_seeds and c["n_links"] == int((other.clink_up >= 0).sum())
    trk.close()


@pytest.mark.parametrize("name", ["single_sector", "semicentral"])
def test_k4_k5_on_the_oracles_cleaned_links(trk_mod, gen_mod, oracle_mod, name):
    """K4 + K5 (+ K6) on cleaned links that are NOT what K3 would make of the links in the work space."""
    ev = gen_mod.generate(name)
    other = _oracle(oracle_mod, gen_mod, ev, nf_dmax=0.05, nf_w0=0.2)
    trk = make_tracker(trk_mod, gen_mod, ev)
    trk.tpc_track_event(ev_dict(ev, True))
    own_links = trk.tpc_debug_get("link_up")
    trk.tpc_debug_inject("clink_up", other.clink_up)
    trk.tpc_debug_inject("clink_dn", other.clink_dn)
    out = trk.tpc_debug_resume("seeds")[0]
    assert np.array_equal(trk.tpc_debug_get("link_up"), own_links)          # K2 / K3 did not run again
    assert np.array_equal(trk.tpc_debug_get("start_hit"), other.start_hit)
    rows = trk.tpc_debug_get("tl_rows")
    assert np.array_equal(trk.tpc_debug_get("tl_table"), other.tl_table)
    assert np.array_equal(rows[:, 2], other.tl_n_hits) and np.array_equal(rows[:, 0], other.tl_first_row)
    built = other.tl_n_hits > 0
    par = trk.tpc_debug_get("tl_par")[built]
    refp = np.concatenate([other.tl_par, other.tl_chi2[:, None]], axis=1)[built]
    assert (np.abs(par - refp) / np.maximum(1.0, np.abs(refp))).max() <= TOL
    _tracks_equal(trk.to_numpy(out), other)
    trk.close()


@pytest.mark.parametrize("name", ["single_sector", "semicentral"])
def test_k6_on_the_oracles_tracklets(trk_mod, gen_mod, oracle_mod, name):
    """K6 alone on the tracklets of an oracle run whose constructor had other gates (same start hits)."""
    ev = gen_mod.generate(name)
    other = _oracle(oracle_mod, gen_mod, ev, chi2_ext=6.0, max_gap=2, chi2_link=12.0)    # O5 differs; O2-O4, O6 identical
    own = _oracle(oracle_mod, gen_mod, ev)
    assert np.array_equal(other.start_hit, own.start_hit) and not np.array_equal(other.tl_table, own.tl_table)
    trk = make_tracker(trk_mod, gen_mod, ev)
    trk.tpc_track_event(ev_dict(ev, True))
    trk.tpc_debug_inject("tl_rows", np.stack([other.tl_first_row, other.tl_last_row, other.tl_n_hits], axis=1))
    trk.tpc_debug_inject("tl_par", np.concatenate([other.tl_par, other.tl_chi2[:, None]], axis=1))
    trk.tpc_debug_inject("tl_table", other.tl_table)
    assert np.array_equal(trk.tpc_debug_get("tl_table"), other.tl_table)    # the injection reads back
    out = trk.tpc_debug_resume("select")[0]
    _tracks_equal(trk.to_numpy(out), other)
    assert trk.tpc_get_counters()["n_row_visits"] == 0                      # K5 did not run again
    trk.close()


def test_k5_alone_runs_again_on_the_work_space(trk_mod, gen_mod, oracle_mod):
    ev = gen_mod.generate("semicentral")
    ref = _oracle(oracle_mod, gen_mod, ev)
    trk = make_tracker(trk_mod, gen_mod, ev)
    trk.tpc_track_event(ev_dict(ev, True))
    garbage = np.full_like(ref.tl_table, -1)
    trk.tpc_debug_inject("tl_table", garbage)
    out = trk.tpc_debug_resume("construct")[0]
    assert np.array_equal(trk.tpc_debug_get("tl_table"), ref.tl_table)
    _tracks_equal(trk.to_numpy(out), ref)
    trk.close()


def test_inject_and_resume_argument_checks(trk_mod, gen_mod):
    ev = gen_mod.generate("pp")
    trk = make_tracker(trk_mod, gen_mod, ev)
    with pytest.raises(trk_mod.TpcError):                                   # nothing has run
        trk.tpc_debug_resume("clean")
    trk.tpc_track_event(ev_dict(ev, False))
    with pytest.raises(trk_mod.TpcError):                                   # host inputs
        trk.tpc_debug_inject("link_up", np.full(ev.n_clusters, -1, np.int32))
    trk.tpc_track_event(ev_dict(ev, True))
    with pytest.raises(trk_mod.TpcError):                                   # wrong size
        trk.tpc_debug_inject("link_up", np.full(ev.n_clusters - 1, -1, np.int32))
    with pytest.raises(trk_mod.TpcError):                                   # a hit index outside the event
        trk.tpc_debug_inject("link_up", np.full(ev.n_clusters, ev.n_clusters, np.int32))
    with pytest.raises(trk_mod.TpcError):                                   # not injectable
        trk.tpc_debug_inject("start_hit", trk.tpc_debug_get("start_hit"))
    trk.tpc_debug_inject("link_up", np.full(ev.n_clusters, -1, np.int32))   # no links at all: no tracks
    out = trk.tpc_debug_resume("clean")[0]
    assert out.n_tracks == 0 and trk.tpc_get_counters()["n_seeds"] == 0
    trk.close()


# ---------------------------------------------------------------------------------------------------------
# checked mode
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("device", [True, False])
def test_checked_mode(trk_mod, gen_mod, oracle_mod, device):
    import torch
    ev = gen_mod.generate("pp")
    ref = _oracle(oracle_mod, gen_mod, ev)
    p = trk_mod.tpc_default_params(); p.checked = 1
    trk = make_tracker(trk_mod, gen_mod, ev, params=p)

    def run(x=None, y=None):
        d = dict(sector_offset=ev.sector_offset, y=ev.y if y is None else y, z=ev.z, row=ev.row)
        if x is not None:
            d["x"] = x
        if device:
            d = {k: (torch.from_numpy(np.ascontiguousarray(a)).cuda() if k != "sector_offset" else a) for k, a in d.items()}
        return trk.tpc_track_event(d)

    for x in (None, ev.x, ev.x + np.float32(5e-4)):                        # no x, exact x, x within 1e-3 cm
        out = run(x=x)
        assert np.array_equal(trk.to_numpy(out)["hit_idx"], ref.hit_idx)
    bad_x = ev.x.copy(); bad_x[ev.n_clusters // 2] += np.float32(2e-3)
    with pytest.raises(trk_mod.TpcError) as ei:
        run(x=bad_x)
    assert ei.value.status == trk_mod.TPC_ERR_ARG
    for v in (np.nan, np.inf, -np.inf):
        bad_y = ev.y.copy(); bad_y[7] = v
        with pytest.raises(trk_mod.TpcError) as ei:
            run(y=bad_y)
        assert ei.value.status == trk_mod.TPC_ERR_ARG
    assert np.array_equal(trk.to_numpy(run())["hit_idx"], ref.hit_idx)       # the tracker is fine afterwards
    trk.close()
    # fast mode: the same inputs are not checked (x ignored); non-finite coordinates must not fault the device
    fast = make_tracker(trk_mod, gen_mod, ev)
    d = dict(sector_offset=ev.sector_offset, x=bad_x, y=ev.y, z=ev.z, row=ev.row)
    assert np.array_equal(fast.to_numpy(fast.tpc_track_event(d))["hit_idx"], ref.hit_idx)
    bad_y = ev.y.copy(); bad_y[::97] = np.nan
    fast.tpc_track_event(dict(sector_offset=ev.sector_offset, y=bad_y, z=ev.z, row=ev.row))   # undefined tracks, no fault
    assert np.array_equal(fast.to_numpy(fast.tpc_track_event(dict(sector_offset=ev.sector_offset, y=ev.y, z=ev.z, row=ev.row)))["hit_idx"],
                          ref.hit_idx)
    fast.close()
    # the oracle's checked mode rejects the same coordinates
    po = oracle_mod.default_params(); po.checked = 1
    with pytest.raises(ValueError):
        oracle_mod.track_event(make_geometry(oracle_mod, gen_mod, ev), ev.sector_offset, bad_y, ev.z, ev.row, params=po)


# ---------------------------------------------------------------------------------------------------------
# corner cases of the boundary (round-1 review)
# ---------------------------------------------------------------------------------------------------------
def test_device_outputs_of_a_ticket_survive_the_next_submit(trk_mod, gen_mod):
    """submit A, submit B, wait A, submit C (which runs in the work space A used), wait B, wait C: A's DEVICE outputs
    are still A's (each ticket owns its output arrays; they are handed over at the wait)."""
    evs = [gen_mod.generate("semicentral", e) for e in range(3)]
    trk = make_tracker(trk_mod, gen_mod, evs[0])
    ref = make_tracker(trk_mod, gen_mod, evs[0])
    want = [ref.to_numpy(ref.tpc_track_event(ev_dict(ev, True))) for ev in evs]
    d = [[ev_dict(ev, True)] for ev in evs]
    ta = trk.tpc_submit_events(d[0]); tb = trk.tpc_submit_events(d[1])
    out_a = trk.tpc_wait_events(ta)
    tc = trk.tpc_submit_events(d[2])
    out_b = trk.tpc_wait_events(tb)
    out_c = trk.tpc_wait_events(tc)          # C has run to completion in A's former work space
    for out, w in ((out_a, want[0]), (out_b, want[1]), (out_c, want[2])):
        got = trk.to_numpy(out[0])
        for k in w:
            assert np.array_equal(got[k], w[k]), k
    trk.close(); ref.close()


def test_small_event_after_and_beside_a_central_one(trk_mod, gen_mod, oracle_mod):
    """The selector's chunking follows the largest sector task of the CALL: a tiny event after a central one on the
    same tracker, and both in one batch (where the tiny event's tasks get chunks without any row)."""
    big, small = gen_mod.generate("central"), gen_mod.tiny_sector(n_tracks=3, seed=5, noise_frac=0.1, sigma=0.08, n_sectors=36)
    refs = [_oracle(oracle_mod, gen_mod, ev) for ev in (big, small)]
    trk = make_tracker(trk_mod, gen_mod, big)
    assert np.array_equal(trk.to_numpy(trk.tpc_track_event(ev_dict(big, True)))["hit_idx"], refs[0].hit_idx)
    assert np.array_equal(trk.to_numpy(trk.tpc_track_event(ev_dict(small, True)))["hit_idx"], refs[1].hit_idx)
    outs = trk.tpc_track_events([ev_dict(small, True), ev_dict(big, True), ev_dict(small, True)])
    for o, r in zip(outs, (refs[1], refs[0], refs[1])):
        _tracks_equal(trk.to_numpy(o), r)
    trk.close()


def test_row_capacity_error_on_a_used_tracker(trk_mod, gen_mod, oracle_mod):
    """An over-full pad row is reported as TPC_ERR_CAPACITY -- also when the work space holds an earlier event's
    links (the later kernels do nothing once K1 has rejected the batch) -- and the tracker goes on working."""
    ev = gen_mod.generate("single_sector")
    ref = _oracle(oracle_mod, gen_mod, ev)
    trk = make_tracker(trk_mod, gen_mod, ev)
    for _ in range(2):
        assert np.array_equal(trk.to_numpy(trk.tpc_track_event(ev_dict(ev, True)))["hit_idx"], ref.hit_idx)
        n = 2100
        rng = np.random.default_rng(0)
        with pytest.raises(trk_mod.TpcError) as ei:
            trk.tpc_track_event(dict(sector_offset=np.array([0, n], np.int32), y=rng.uniform(-10, 10, n).astype(np.float32),
                                     z=rng.uniform(0, 200, n).astype(np.float32), row=np.full(n, 7, np.int32)))
        assert ei.value.status == trk_mod.TPC_ERR_CAPACITY
        bad_row = ev.row.copy(); bad_row[3] = 200
        with pytest.raises(trk_mod.TpcError) as ei:
            trk.tpc_track_event(dict(sector_offset=ev.sector_offset, y=ev.y, z=ev.z, row=bad_row))
        assert ei.value.status == trk_mod.TPC_ERR_ARG
    trk.close()
