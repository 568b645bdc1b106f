"""GPU-vs-oracle parity through the C ABI (-m gpu).  Reference = the oracle's strict-float32 mode
(BASELINE.json:5 fixes float32 for the fit; decisions are taken in the kernel's precision on both sides).
Integer results (links, start hits, tracklet tables, track hit lists) must be identical; a mismatch is tolerated
only where the oracle's decision margin is below 1e-5 and is counted.  Parameters and chi2: |d| <= 1e-4*max(1,|v|).
"""
import numpy as np
import pytest

from conftest import make_geometry

pytestmark = pytest.mark.gpu

MARGIN = 1e-5
TOL = 1e-4


@pytest.fixture(scope="module")
def trk_mod():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1712_09416_b200 import tracker
    return tracker


def make_tracker(trk_mod, gen_mod, ev, params=None):
    return trk_mod.Tracker(ev.n_sectors, gen_mod.row_x().astype(np.float32), gen_mod.TAN_HALF_ANGLE, ev.sigma, ev.sigma,
                           ev.bz, params=params)


def ev_dict(ev, device):
    if device:
        import torch
        return dict(sector_offset=ev.sector_offset, y=torch.from_numpy(ev.y).cuda(), z=torch.from_numpy(ev.z).cuda(),
                    row=torch.from_numpy(ev.row).cuda())
    return dict(sector_offset=ev.sector_offset, y=ev.y, z=ev.z, row=ev.row)


def copy_params(oracle_p, trk_mod):
    p = trk_mod.tpc_default_params()
    for name, _ in p._fields_:
        setattr(p, name, getattr(oracle_p, name))
    return p


def compare_event(trk, out, ev, ref, event=0, check_stages=True):
    """Returns the number of tolerated low-margin flips; asserts on everything else."""
    flips = 0
    tainted = np.zeros(ev.n_clusters, bool)
    if check_stages:
        for k in ("link_up", "link_dn"):
            g = trk.tpc_debug_get(k, event)
            bad = g != ref[k]
            assert np.all(ref.nf_margin[bad] < MARGIN), (k, int(bad.sum()), ref.nf_margin[bad].max())
            flips += int(bad.sum()); tainted |= bad
        if flips == 0:
            for k in ("clink_up", "clink_dn"):
                assert np.array_equal(trk.tpc_debug_get(k, event), ref[k]), k
            assert np.array_equal(trk.tpc_debug_get("start_hit", event), ref.start_hit)
            rows = trk.tpc_debug_get("tl_rows", event)
            tab = trk.tpc_debug_get("tl_table", event)
            par = trk.tpc_debug_get("tl_par", event)
            same = (tab == ref.tl_table).all(axis=1)
            bad = ~same
            assert np.all(ref.tl_margin[bad] < MARGIN), (int(bad.sum()), ref.tl_margin[bad].max() if bad.any() else 0)
            flips += int(bad.sum())
            assert np.array_equal(rows[same, 0], ref.tl_first_row[same])
            assert np.array_equal(rows[same, 1], ref.tl_last_row[same])
            assert np.array_equal(rows[same, 2], ref.tl_n_hits[same])
            built = same & (ref.tl_n_hits > 0)     # a start hit skipped by the seed de-duplication (R23) has no fit
            refp = np.concatenate([ref.tl_par, ref.tl_chi2[:, None]], axis=1)[built]
            err = np.abs(par[built] - refp) / np.maximum(1.0, np.abs(refp))
            assert err.max(initial=0.0) <= TOL, err.max()
    res = trk.to_numpy(out)
    if flips == 0:
        assert res["n_tracks"] == ref.n_tracks and res["n_track_hits"] == ref.n_track_hits
        for k in ("trk_sector", "trk_first_hit", "trk_n_hits", "trk_ndf", "hit_idx"):
            assert np.array_equal(res[k], ref[k]), k
        for k in ("trk_x", "trk_y", "trk_z", "trk_sinphi", "trk_tgl", "trk_qpt", "trk_chi2"):
            err = np.abs(res[k] - ref[k]) / np.maximum(1.0, np.abs(ref[k]))
            assert err.max(initial=0.0) <= TOL, (k, err.max())
    else:
        # tolerated flips upstream: tracks must agree except a handful
        assert abs(res["n_tracks"] - ref.n_tracks) <= 4 * flips
    # properties that hold whatever happened
    assert np.unique(res["hit_idx"]).size == res["hit_idx"].size
    return flips, res


@pytest.mark.parametrize("device_inputs", [True, False])
@pytest.mark.parametrize("name", ["single_sector", "pp", "semicentral"])
def test_parity_configs(trk_mod, gen_mod, event_and_oracle, name, device_inputs):
    ev, ref = event_and_oracle(name, "float")
    trk = make_tracker(trk_mod, gen_mod, ev)
    out = trk.tpc_track_event(ev_dict(ev, device_inputs))
    flips, res = compare_event(trk, out, ev, ref)
    assert flips == 0, "strict-float32 arithmetic on both sides: no flips expected"
    c = trk.tpc_get_counters()
    assert c["n_clusters"] == ev.n_clusters and c["n_seeds"] == ref.n_seeds and c["n_tracks"] == ref.n_tracks
    assert c["n_links"] == int((ref.clink_up >= 0).sum()) and c["n_kernel_launches"] >= 10
    assert c["n_tracklets"] == int((ref.tl_n_hits > 0).sum()) < c["n_seeds"]
    trk.close()


@pytest.mark.parametrize("name", ["single_sector", "semicentral"])
def test_parity_without_seed_dedup(trk_mod, gen_mod, oracle_mod, name):
    """seed_dedup = 0: every start hit is fitted (three times the tracklets under way: the constructor runs with
    its large slot count, one CTA per SM)."""
    ev = gen_mod.generate(name)
    po = oracle_mod.default_params(); po.seed_dedup = 0
    ref = oracle_mod.track_event(make_geometry(oracle_mod, gen_mod, ev), ev.sector_offset, ev.y, ev.z, ev.row,
                                 params=po, precision="float")
    trk = make_tracker(trk_mod, gen_mod, ev, params=copy_params(po, trk_mod))
    out = trk.tpc_track_event(ev_dict(ev, True))
    flips, res = compare_event(trk, out, ev, ref)
    assert flips == 0
    c = trk.tpc_get_counters()
    assert c["n_tracklets"] == c["n_seeds"] == ref.n_seeds
    trk.close()


def test_parity_central_full_size(trk_mod, gen_mod, event_and_oracle):
    """BASELINE.json config 4 (the bench workload's event) at full size, every output compared."""
    ev, ref = event_and_oracle("central", "float")
    trk = make_tracker(trk_mod, gen_mod, ev)
    out = trk.tpc_track_event(ev_dict(ev, True))
    flips, res = compare_event(trk, out, ev, ref)
    assert flips == 0
    trk.close()


def test_parity_batch_of_events_matches_single_events(trk_mod, gen_mod, oracle_mod):
    """tpc_track_events: every event of a batch gives what it gives alone (and what the oracle gives)."""
    evs = [gen_mod.generate("semicentral", e) for e in range(3)] + [gen_mod.generate("pp", 0)]
    trk = make_tracker(trk_mod, gen_mod, evs[0])
    outs = trk.tpc_track_events([ev_dict(ev, True) for ev in evs])
    for e, ev in enumerate(evs):
        ref = oracle_mod.track_event(make_geometry(oracle_mod, gen_mod, ev), ev.sector_offset, ev.y, ev.z, ev.row,
                                     precision="float")
        flips, _ = compare_event(trk, outs[e], ev, ref, event=e)
        assert flips == 0
    trk.close()


@pytest.mark.parametrize("per_group,device", [(1, False), (2, False), (0, False), (2, True)])
def test_host_batches_run_as_overlapping_groups(trk_mod, gen_mod, oracle_mod, per_group, device):
    """Host-input batches are cut into groups of events on separate streams (copies of one group overlap the
    kernels of another); 7 events in groups of 1 also cycle the three slots; device-input batches are grouped on
    request.  Results must not depend on it."""
    evs = [gen_mod.generate("pp", e) for e in range(4)] + [gen_mod.generate("semicentral", 0)] + \
          [gen_mod.generate("pp", e) for e in range(4, 6)]
    trk = make_tracker(trk_mod, gen_mod, evs[0])
    trk.tpc_tracker_set_group_events(per_group)
    outs = trk.tpc_track_events([ev_dict(ev, device) for ev in evs])
    res = [trk.to_numpy(o) for o in outs]
    c = trk.tpc_get_counters()
    assert c["n_events"] == len(evs) and c["n_clusters"] == sum(ev.n_clusters for ev in evs)
    assert c["n_tracks"] == sum(r["n_tracks"] for r in res)
    for e, ev in enumerate(evs):
        ref = oracle_mod.track_event(make_geometry(oracle_mod, gen_mod, ev), ev.sector_offset, ev.y, ev.z, ev.row,
                                     precision="float")
        assert res[e]["n_tracks"] == ref.n_tracks
        for k in ("trk_sector", "trk_first_hit", "trk_n_hits", "trk_ndf", "hit_idx"):
            assert np.array_equal(res[e][k], ref[k]), (e, k)
        for k in ("trk_y", "trk_z", "trk_sinphi", "trk_tgl", "trk_qpt", "trk_chi2"):
            err = np.abs(res[e][k] - ref[k]) / np.maximum(1.0, np.abs(ref[k]))
            assert err.max(initial=0.0) <= TOL, (e, k, err.max())
    if per_group == 1:   # events of the last three groups keep their intermediates, earlier ones do not
        assert np.array_equal(trk.tpc_debug_get("start_hit", 6), ref.start_hit)
        with pytest.raises(trk_mod.TpcError):
            trk.tpc_debug_get("start_hit", 0)
    trk.close()


@pytest.mark.parametrize("step", [1, 2])
def test_parity_link_step_and_dense_rows(trk_mod, gen_mod, oracle_mod, step):
    p = oracle_mod.default_params()
    p.link_step = step
    p.nf_dmax = 1.0
    for seed, ntr, noise in ((7, 6, 0.5), (8, 12, 1.0), (9, 25, 3.0)):
        ev = gen_mod.tiny_sector(n_tracks=ntr, seed=seed, noise_frac=noise)
        ref = oracle_mod.track_event(make_geometry(oracle_mod, gen_mod, ev), ev.sector_offset, ev.y, ev.z, ev.row,
                                     params=p, precision="float")
        trk = make_tracker(trk_mod, gen_mod, ev, params=copy_params(p, trk_mod))
        out = trk.tpc_track_event(ev_dict(ev, False))
        flips, _ = compare_event(trk, out, ev, ref)
        assert flips == 0
        trk.close()


def test_coincident_hits_and_ties(trk_mod, gen_mod, oracle_mod):
    """S22: duplicated clusters (identical y, z) -> every tie resolved towards the lowest caller index."""
    ev = gen_mod.tiny_sector(n_tracks=10, seed=3, noise_frac=0.2)
    dup = np.arange(0, ev.n_clusters, 3)
    y = np.concatenate([ev.y, ev.y[dup]]); z = np.concatenate([ev.z, ev.z[dup]]); row = np.concatenate([ev.row, ev.row[dup]])
    ev2 = gen_mod.Event(1, np.array([0, y.size], np.int32), gen_mod.row_x()[row].astype(np.float32), y, z, row,
                        np.concatenate([ev.label, ev.label[dup]]), ev.tracks, sigma=ev.sigma)
    ref = oracle_mod.track_event(make_geometry(oracle_mod, gen_mod, ev2), ev2.sector_offset, y, z, row, precision="float")
    trk = make_tracker(trk_mod, gen_mod, ev2)
    out = trk.tpc_track_event(ev_dict(ev2, False))
    flips, _ = compare_event(trk, out, ev2, ref)
    assert flips == 0
    trk.close()


def test_degenerate_inputs(trk_mod, gen_mod):
    rx = gen_mod.row_x().astype(np.float32)
    trk = trk_mod.Tracker(36, rx, gen_mod.TAN_HALF_ANGLE, 0.06, 0.06, 0.5)
    z = np.zeros(0, np.float32)
    out = trk.tpc_track_event(dict(sector_offset=np.zeros(37, np.int32), y=z, z=z, row=np.zeros(0, np.int32)))
    assert out.n_tracks == 0 and out.n_track_hits == 0
    so = np.zeros(37, np.int32); so[4:] = 2
    out = trk.tpc_track_event(dict(sector_offset=so, y=np.array([0, 0.1], np.float32), z=np.array([10, 10.1], np.float32),
                                   row=np.array([5, 6], np.int32)))
    assert out.n_tracks == 0
    assert np.all(trk.tpc_debug_get("link_up") == -1)
    # errors: row out of range, bad sector_offset
    with pytest.raises(trk_mod.TpcError) as ei:
        trk.tpc_track_event(dict(sector_offset=so, y=np.zeros(2, np.float32), z=np.zeros(2, np.float32),
                                 row=np.array([5, 159], np.int32)))
    assert ei.value.status == trk_mod.TPC_ERR_ARG
    bad = so.copy(); bad[3] = 5
    with pytest.raises(trk_mod.TpcError):
        trk.tpc_track_event(dict(sector_offset=bad, y=np.zeros(2, np.float32), z=np.zeros(2, np.float32),
                                 row=np.array([5, 6], np.int32)))
    # the tracker is still usable after an error
    ev = gen_mod.generate("pp")
    out = trk.tpc_track_event(ev_dict(ev, False))
    assert out.n_tracks > 50
    trk.close()


def test_row_capacity_error(trk_mod, gen_mod):
    rx = gen_mod.row_x().astype(np.float32)
    trk = trk_mod.Tracker(1, rx, gen_mod.TAN_HALF_ANGLE, 0.06, 0.06, 0.5)
    n = 2100   # > TPC_MAX_ROW_HITS in one (sector,row)
    rng = np.random.default_rng(0)
    with pytest.raises(trk_mod.TpcError) as ei:
        trk.tpc_track_event(dict(sector_offset=np.array([0, n], np.int32), y=rng.uniform(-10, 10, n).astype(np.float32),
                                 z=rng.uniform(0, 200, n).astype(np.float32), row=np.full(n, 7, np.int32)))
    assert ei.value.status == trk_mod.TPC_ERR_CAPACITY
    trk.close()


def test_seed_pool_grows(trk_mod, gen_mod, oracle_mod):
    """16k isolated 5-hit chains: one start hit per 5 clusters exceeds the default tracklet pool (N/8 + 4096);
    the library must grow the pool, re-run, and still match the oracle."""
    rx = gen_mod.row_x().astype(np.float32)
    n_chain, groups, cols = 16000, 31, 6
    j = np.arange(n_chain)
    g = j % groups; k = (j // groups) % cols; m = j // (groups * cols)
    y0 = -12.0 + 4.0 * k + 2.0 * (g % 2)
    z0 = 2.0 + 2.9 * m
    row = (5 * g[:, None] + np.arange(5)[None, :]).reshape(-1).astype(np.int32)
    y = np.repeat(y0, 5).astype(np.float32); z = np.repeat(z0, 5).astype(np.float32)
    perm = np.random.default_rng(1).permutation(row.size)
    y, z, row = y[perm], z[perm], row[perm]
    ev = gen_mod.Event(1, np.array([0, row.size], np.int32), rx[row], y, z, row, np.zeros(row.size, np.int32),
                       np.zeros((1, 8)), sigma=0.06)
    p = oracle_mod.default_params()
    p.min_tracklet_hits = 4; p.min_track_hits = 4
    ref = oracle_mod.track_event(make_geometry(oracle_mod, gen_mod, ev), ev.sector_offset, y, z, row, params=p,
                                 precision="float")
    assert n_chain >= ref.n_seeds > row.size // 8 + 4096      # outer rows (wider pitch) merge a few chains
    trk = make_tracker(trk_mod, gen_mod, ev, params=copy_params(p, trk_mod))
    out = trk.tpc_track_event(ev_dict(ev, True))
    assert trk.tpc_get_counters()["n_retries"] >= 1
    res = trk.to_numpy(out)
    assert res["n_tracks"] == ref.n_tracks and np.array_equal(res["hit_idx"], ref.hit_idx)
    assert np.array_equal(trk.tpc_debug_get("start_hit"), ref.start_hit)
    assert np.array_equal(trk.tpc_debug_get("tl_table"), ref.tl_table)
    trk.close()


@pytest.mark.parametrize("name,step", [("single_sector", 1), ("semicentral", 1), ("semicentral", 2), ("central", 1)])
def test_refit_parity(trk_mod, gen_mod, oracle_mod, name, step):
    """O8 (tpc_params.refit = 1): refit of every output track over its final hit list; hit lists unchanged,
    parameters / chi2 / ndf / reference row those of the oracle's refit (strict float32)."""
    ev = gen_mod.generate(name)
    p = oracle_mod.default_params()
    p.refit = 1; p.link_step = step
    ref = oracle_mod.track_event(make_geometry(oracle_mod, gen_mod, ev), ev.sector_offset, ev.y, ev.z, ev.row,
                                 params=p, precision="float")
    trk = make_tracker(trk_mod, gen_mod, ev, params=copy_params(p, trk_mod))
    out = trk.tpc_track_event(ev_dict(ev, True))
    flips, res = compare_event(trk, out, ev, ref, check_stages=False)
    assert flips == 0
    c = trk.tpc_get_counters()
    assert c["n_refit_visits"] > 2 * (c["n_track_hits"] - c["n_tracks"]) * 0.9
    # the refit makes hit list and fit consistent: ndf counts the hits of the list (no transport failure here)
    assert np.mean(res["trk_ndf"] == 2 * res["trk_n_hits"] - 5) > 0.99
    base = make_tracker(trk_mod, gen_mod, ev, params=copy_params(oracle_mod.default_params(), trk_mod)) if step == 1 else None
    if base is not None:   # refit off: same hit lists, different parameters
        r0 = base.to_numpy(base.tpc_track_event(ev_dict(ev, True)))
        assert np.array_equal(r0["hit_idx"], res["hit_idx"]) and not np.array_equal(r0["trk_qpt"], res["trk_qpt"])
        assert base.tpc_get_counters()["n_refit_visits"] == 0
        base.close()
    trk.close()


def test_refit_in_a_batch_matches_single_events(trk_mod, gen_mod, oracle_mod):
    evs = [gen_mod.generate("pp", 0), gen_mod.generate("semicentral", 0), gen_mod.generate("pp", 1)]
    p = oracle_mod.default_params()
    p.refit = 1
    trk = make_tracker(trk_mod, gen_mod, evs[0], params=copy_params(p, trk_mod))
    outs = trk.tpc_track_events([ev_dict(ev, False) for ev in evs])
    for ev, o in zip(evs, outs):
        ref = oracle_mod.track_event(make_geometry(oracle_mod, gen_mod, ev), ev.sector_offset, ev.y, ev.z, ev.row,
                                     params=p, precision="float")
        res = trk.to_numpy(o)
        assert np.array_equal(res["hit_idx"], ref.hit_idx) and np.array_equal(res["trk_ndf"], ref.trk_ndf)
        for k in ("trk_x", "trk_y", "trk_z", "trk_sinphi", "trk_tgl", "trk_qpt", "trk_chi2"):
            err = np.abs(res[k] - ref[k]) / np.maximum(1.0, np.abs(ref[k]))
            assert err.max(initial=0.0) <= TOL, (k, err.max())
    trk.close()


@pytest.mark.parametrize("name,device", [("pp", True), ("semicentral", True), ("semicentral", False), ("central", True)])
def test_merge_parity(trk_mod, gen_mod, oracle_mod, name, device):
    """O9 (tpc_params.merge = 1): links between the segments of one particle across sector borders, and the refit's
    outer states they are made from, against the oracle (strict float32)."""
    ev = gen_mod.generate(name)
    p = oracle_mod.default_params()
    p.refit = 1; p.merge = 1
    ref = oracle_mod.track_event(make_geometry(oracle_mod, gen_mod, ev), ev.sector_offset, ev.y, ev.z, ev.row,
                                 params=p, precision="float")
    trk = make_tracker(trk_mod, gen_mod, ev, params=copy_params(p, trk_mod))
    out = trk.tpc_track_event(ev_dict(ev, device))
    flips, res = compare_event(trk, out, ev, ref, check_stages=False)
    assert flips == 0
    outer = np.stack([res[k] for k in ("trk_out_x", "trk_out_y", "trk_out_z", "trk_out_sinphi", "trk_out_tgl",
                                       "trk_out_qpt")], axis=1)
    err = np.abs(outer - ref.trk_out) / np.maximum(1.0, np.abs(ref.trk_out))
    assert err.max(initial=0.0) <= TOL, err.max()
    assert np.array_equal(res["trk_next"], ref.trk_next) and np.array_equal(res["trk_prev"], ref.trk_prev)
    assert np.array_equal(res["trk_global"], ref.trk_global)
    assert (res["trk_next"] >= 0).sum() >= (40 if name == "pp" else 1000)
    # O10: the fit of every global track over all its segments
    for k in ("trk_g_ndf", "trk_g_n_hits", "trk_g_sector"):
        assert np.array_equal(res[k], ref[k]), k
    gfit = np.stack([res[k] for k in ("trk_g_x", "trk_g_y", "trk_g_z", "trk_g_sinphi", "trk_g_tgl", "trk_g_qpt",
                                      "trk_g_chi2")], axis=1)
    err = np.abs(gfit - ref.trk_g) / np.maximum(1.0, np.abs(ref.trk_g))
    assert err.max(initial=0.0) <= TOL, err.max()
    chains = (ref.trk_prev < 0) & (ref.trk_next >= 0)
    more = res["trk_g_n_hits"][chains] > res["trk_n_hits"][chains]      # more hits than the first segment alone
    assert more.mean() > 0.9                                            # (a failed turn at a border ends a pass early)
    trk.close()


def test_merge_in_a_batch_and_argument_checks(trk_mod, gen_mod, oracle_mod):
    evs = [gen_mod.generate("pp", 0), gen_mod.generate("semicentral", 0), gen_mod.generate("pp", 1)]
    p = oracle_mod.default_params()
    p.refit = 1; p.merge = 1
    trk = make_tracker(trk_mod, gen_mod, evs[0], params=copy_params(p, trk_mod))
    for device in (True, False):
        outs = trk.tpc_track_events([ev_dict(ev, device) for ev in evs])
        for ev, o in zip(evs, outs):
            ref = oracle_mod.track_event(make_geometry(oracle_mod, gen_mod, ev), ev.sector_offset, ev.y, ev.z, ev.row,
                                         params=p, precision="float")
            res = trk.to_numpy(o)
            assert np.array_equal(res["trk_next"], ref.trk_next) and np.array_equal(res["trk_prev"], ref.trk_prev)
            assert np.array_equal(res["trk_global"], ref.trk_global)
    trk.close()
    # without refit / merge the extra outputs are absent; merge without refit is refused
    t0 = make_tracker(trk_mod, gen_mod, evs[0])
    r0 = t0.to_numpy(t0.tpc_track_event(ev_dict(evs[0], True)))
    assert "trk_next" not in r0 and "trk_out_x" not in r0
    t0.close()
    q = copy_params(oracle_mod.default_params(), trk_mod)
    q.merge = 1
    with pytest.raises(trk_mod.TpcError):
        make_tracker(trk_mod, gen_mod, evs[0], params=q)
    # a single-sector geometry has no neighbours: no links
    ev1 = gen_mod.generate("single_sector")
    t1 = make_tracker(trk_mod, gen_mod, ev1, params=copy_params(p, trk_mod))
    r1 = t1.to_numpy(t1.tpc_track_event(ev_dict(ev1, True)))
    assert np.all(r1["trk_next"] == -1) and np.all(r1["trk_prev"] == -1)
    assert np.array_equal(r1["trk_global"], np.arange(r1["n_tracks"]))
    t1.close()


def test_parity_config5_in_the_bench_configuration(trk_mod, gen_mod, oracle_mod):
    """BASELINE.json config 5 at full size (16 central events, 29.7 M clusters) launched as bench.py launches it
    (one call, device-resident inputs, work space reserved at create): three sampled events compared with the oracle
    output by output, and counts that hold for the whole batch."""
    import bench
    evs = bench.make_events("central", 16)
    n_total = sum(ev.n_clusters for ev in evs)
    trk = trk_mod.Tracker(evs[0].n_sectors, gen_mod.row_x().astype(np.float32), gen_mod.TAN_HALF_ANGLE, evs[0].sigma,
                          evs[0].sigma, evs[0].bz, max_events=len(evs), max_clusters=n_total)
    outs = trk.tpc_track_events([ev_dict(ev, True) for ev in evs])
    c = trk.tpc_get_counters()
    assert c["n_events"] == 16 and c["n_clusters"] == n_total and c["n_retries"] == 0
    assert c["n_tracks"] == sum(o.n_tracks for o in outs) and c["n_track_hits"] == sum(o.n_track_hits for o in outs)
    for e in (0, 7, 15):
        ev = evs[e]
        ref = oracle_mod.track_event(make_geometry(oracle_mod, gen_mod, ev), ev.sector_offset, ev.y, ev.z, ev.row,
                                     precision="float")
        flips, res = compare_event(trk, outs[e], ev, ref, event=e)
        assert flips == 0
    for o in outs:   # every event: a hit is in at most one track
        h = trk.to_numpy(o)["hit_idx"]
        assert np.unique(h).size == h.size
    trk.close()


@pytest.mark.parametrize("n_tracks,refit", [(800, 0), (1300, 1)])
def test_parity_rows_larger_than_the_shared_memory_stages(trk_mod, gen_mod, oracle_mod, n_tracks, refit):
    """Pad rows of 500-1500 clusters: more than the neighbour finder (640) and the sweep constructor (640) stage in
    shared memory, so their read-in-place paths run (mixed with staged rows), still below TPC_MAX_ROW_HITS."""
    r = gen_mod.Recipe("dense", n_sectors=1, n_primaries=n_tracks, pt_mode=0, pt_a=0.4, pt_b=4.0, sigma=0.06,
                       inefficiency=0.02, noise_frac=0.2, bz=0.5, config_id=60)
    ev = gen_mod.generate(r, event=0)
    cnt = np.bincount(ev.row, minlength=159)
    assert cnt.max() > 800 and cnt.max() < 2048 and cnt.min() < 1000
    p = oracle_mod.default_params()
    p.refit = refit
    ref = oracle_mod.track_event(make_geometry(oracle_mod, gen_mod, ev), ev.sector_offset, ev.y, ev.z, ev.row,
                                 params=p, precision="float")
    trk = make_tracker(trk_mod, gen_mod, ev, params=copy_params(p, trk_mod))
    out = trk.tpc_track_event(ev_dict(ev, True))
    flips, res = compare_event(trk, out, ev, ref, check_stages=(refit == 0))
    assert flips == 0 and res["n_tracks"] > 500
    trk.close()


@pytest.mark.parametrize("n_rows", [37, 64])
def test_parity_other_row_counts(trk_mod, gen_mod, oracle_mod, n_rows):
    """Geometry is an input: a TPC of 37 or 64 pad rows (not multiples of 8 / 32), refit and merge on."""
    ev = gen_mod.generate("semicentral")
    keep = ev.row < n_rows
    so = np.concatenate([[0], np.cumsum([keep[ev.sector_offset[s]:ev.sector_offset[s + 1]].sum()
                                         for s in range(ev.n_sectors)])]).astype(np.int32)
    y, z, row = ev.y[keep].copy(), ev.z[keep].copy(), ev.row[keep].copy()
    rx = gen_mod.row_x().astype(np.float32)[:n_rows].copy()
    p = oracle_mod.default_params()
    p.refit = 1; p.merge = 1
    g = oracle_mod.Geometry(ev.n_sectors, rx, gen_mod.TAN_HALF_ANGLE, ev.sigma, ev.sigma, ev.bz)
    ref = oracle_mod.track_event(g, so, y, z, row, params=p, precision="float")
    trk = trk_mod.Tracker(ev.n_sectors, rx, gen_mod.TAN_HALF_ANGLE, ev.sigma, ev.sigma, ev.bz, params=copy_params(p, trk_mod))
    import torch
    out = trk.tpc_track_event(dict(sector_offset=so, y=torch.from_numpy(y).cuda(), z=torch.from_numpy(z).cuda(),
                                   row=torch.from_numpy(row).cuda()))
    res = trk.to_numpy(out)
    assert ref.n_tracks > 500 and res["n_tracks"] == ref.n_tracks
    for k in ("trk_sector", "trk_first_hit", "trk_n_hits", "trk_ndf", "hit_idx", "trk_next", "trk_prev", "trk_global"):
        assert np.array_equal(res[k], ref[k]), k
    for k in ("trk_x", "trk_y", "trk_z", "trk_sinphi", "trk_tgl", "trk_qpt", "trk_chi2"):
        err = np.abs(res[k] - ref[k]) / np.maximum(1.0, np.abs(ref[k]))
        assert err.max(initial=0.0) <= TOL, (k, err.max())
    assert np.array_equal(trk.tpc_debug_get("start_hit", 0), ref.start_hit)
    trk.close()


@pytest.mark.parametrize("device", [True, False])
def test_submit_wait_gives_what_the_sync_call_gives(trk_mod, gen_mod, oracle_mod, device):
    """tpc_submit_events / tpc_wait_events: three batches in flight, results those of tpc_track_events (refit and
    merge on); a fourth submit and a wait on an idle ticket are refused."""
    p = oracle_mod.default_params()
    p.refit = 1; p.merge = 1
    batches = [[gen_mod.generate("pp", 0), gen_mod.generate("semicentral", 0)],
               [gen_mod.generate("semicentral", 1)], [gen_mod.generate("pp", 1), gen_mod.generate("pp", 2)],
               [gen_mod.generate("semicentral", 2), gen_mod.generate("pp", 3)]]
    trk = make_tracker(trk_mod, gen_mod, batches[0][0], params=copy_params(p, trk_mod))
    ref_trk = make_tracker(trk_mod, gen_mod, batches[0][0], params=copy_params(p, trk_mod))
    dicts = [[ev_dict(ev, device) for ev in b] for b in batches]
    t0 = trk.tpc_submit_events(dicts[0])
    t1 = trk.tpc_submit_events(dicts[1])
    t2 = trk.tpc_submit_events(dicts[2])
    assert {t0, t1, t2} == {0, 1, 2}
    with pytest.raises(trk_mod.TpcError):
        trk.tpc_submit_events(dicts[3])               # three in flight already
    got = {0: [trk.to_numpy(o) for o in trk.tpc_wait_events(t0)]}
    t3 = trk.tpc_submit_events(dicts[3])               # the freed ticket is handed out again
    assert t3 == t0
    got[1] = [trk.to_numpy(o) for o in trk.tpc_wait_events(t1)]
    got[2] = [trk.to_numpy(o) for o in trk.tpc_wait_events(t2)]
    got[3] = [trk.to_numpy(o) for o in trk.tpc_wait_events(t3)]
    for k, b in enumerate(batches):
        want = [ref_trk.to_numpy(o) for o in ref_trk.tpc_track_events(dicts[k])]
        for e, ev in enumerate(b):
            assert got[k][e]["n_tracks"] == want[e]["n_tracks"] > 50
            for name in want[e]:
                assert np.array_equal(got[k][e][name], want[e][name]), (k, e, name)
    ref = oracle_mod.track_event(make_geometry(oracle_mod, gen_mod, batches[1][0]), batches[1][0].sector_offset,
                                 batches[1][0].y, batches[1][0].z, batches[1][0].row, params=p, precision="float")
    assert np.array_equal(got[1][0]["hit_idx"], ref.hit_idx) and np.array_equal(got[1][0]["trk_next"], ref.trk_next)
    with pytest.raises(trk_mod.TpcError):
        lib_out = (trk_mod.tpc_event_out * 1)()
        trk_mod._check(trk_mod.lib.tpc_wait_events(trk._h, 0, lib_out))     # nothing in flight
    trk.close(); ref_trk.close()


def test_parity_central_link_step_2_full_size(trk_mod, gen_mod, oracle_mod):
    """BASELINE.json config 4 with Delta = 2, every stage and every output compared."""
    ev = gen_mod.generate("central")
    po = oracle_mod.default_params(); po.link_step = 2
    ref = oracle_mod.track_event(make_geometry(oracle_mod, gen_mod, ev), ev.sector_offset, ev.y, ev.z, ev.row,
                                 params=po, precision="float")
    trk = make_tracker(trk_mod, gen_mod, ev, params=copy_params(po, trk_mod))
    out = trk.tpc_track_event(ev_dict(ev, True))
    flips, res = compare_event(trk, out, ev, ref)
    assert flips == 0 and res["n_tracks"] > 20000
    trk.close()


def test_parity_dense_workload(trk_mod, gen_mod, oracle_mod):
    """The bench's second workload (2.5 x central multiplicity, 4.6 M clusters, pad rows of up to ~1000 hits: beyond
    the 640 hits K2 / K5 stage in shared memory, read in place), every stage and every output compared."""
    ev = gen_mod.generate("dense")
    ref = oracle_mod.track_event(make_geometry(oracle_mod, gen_mod, ev), ev.sector_offset, ev.y, ev.z, ev.row,
                                 precision="float")
    trk = make_tracker(trk_mod, gen_mod, ev)
    out = trk.tpc_track_event(ev_dict(ev, True))
    flips, res = compare_event(trk, out, ev, ref)
    assert flips == 0 and res["n_tracks"] > 50000
    c = trk.tpc_get_counters()
    assert c["n_tracklets"] == int((ref.tl_n_hits > 0).sum())
    trk.close()
