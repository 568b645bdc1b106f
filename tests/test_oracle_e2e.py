"""Pins of the oracle's tracklet tables (O5 bookkeeping), selector (O6), output (O7) and end-to-end physics
(SURVEY.md 8(c).5 "O6" and "End-to-end"): structural invariants, a brute-force owner computed here from the
tracklet tables, and stated efficiency / fake-rate thresholds against generator truth."""
import numpy as np
import pytest

from evaluate import efficiency


@pytest.mark.parametrize("name", ["single_sector", "pp", "semicentral"])
def test_tracklet_tables_are_consistent(event_and_oracle, name):
    ev, res = event_and_oracle(name, "float")
    sector = np.repeat(np.arange(ev.n_sectors), np.diff(ev.sector_offset))
    tab = res.tl_table
    S, NR = tab.shape
    assert S == res.n_seeds == res.start_hit.size
    has = tab >= 0
    assert np.array_equal(has.sum(axis=1), res.tl_n_hits)
    rows = np.arange(NR)[None, :]
    first = np.where(has, rows, NR).min(axis=1); last = np.where(has, rows, -1).max(axis=1)
    built = res.tl_n_hits > 0       # a start hit skipped by the seed de-duplication (R23) builds nothing
    assert np.array_equal(first[built], res.tl_first_row[built]) and np.array_equal(last[built], res.tl_last_row[built])
    assert np.all(res.tl_first_row[~built] == -1) and np.all(res.tl_last_row[~built] == -1)
    assert 0.15 * S < built.sum() < 0.75 * S
    # a table entry of row r is a hit of row r in the seed's sector
    ti, ri = np.nonzero(has)
    assert np.array_equal(ev.row[tab[ti, ri]], ri)
    seed_sector = np.repeat(np.arange(ev.n_sectors), np.diff(res.seed_offset))
    assert np.array_equal(sector[tab[ti, ri]], seed_sector[ti])
    assert np.all(res.tl_n_hits[built] >= 1)
    assert np.all(np.isfinite(res.tl_par))
    good = res.tl_n_hits >= 10          # a 2-3 hit stub may end on an update that pushes |sin phi| past 1
    assert np.all(np.abs(res.tl_par[good, 2]) < 1.0)
    assert np.all(res.tl_chi2 >= 0)


@pytest.mark.parametrize("name", ["single_sector", "pp", "semicentral"])
def test_selector_equals_brute_force_owner(oracle_mod, event_and_oracle, name):
    ev, res = event_and_oracle(name, "float")
    p = oracle_mod.default_params()
    tab, nh = res.tl_table, res.tl_n_hits
    owner = {}
    for i in range(res.n_seeds):                  # ascending canonical id: ties keep the lower id
        if nh[i] < p.min_tracklet_hits:
            continue
        for h in tab[i][tab[i] >= 0]:
            o = owner.get(int(h))
            if o is None or nh[i] > nh[o]:
                owner[int(h)] = i
    exp_seed, exp_hits = [], []
    for i in range(res.n_seeds):
        if nh[i] < p.min_tracklet_hits:
            continue
        mine = [int(h) for h in tab[i] if h >= 0 and owner[int(h)] == i]   # row ascending
        if len(mine) >= p.min_track_hits:
            exp_seed.append(i); exp_hits.append(mine)
    assert np.array_equal(res.trk_seed, np.array(exp_seed, np.int32))
    assert np.array_equal(res.trk_n_hits, [len(h) for h in exp_hits])
    assert np.array_equal(res.hit_idx, np.concatenate(exp_hits) if exp_hits else np.zeros(0, np.int32))
    assert np.array_equal(res.trk_first_hit, np.concatenate([[0], np.cumsum(res.trk_n_hits)[:-1]]))
    # invariants: a hit belongs to at most one track; params are the tracklet's, unchanged
    assert np.unique(res.hit_idx).size == res.hit_idx.size
    sd = res.trk_seed
    assert np.array_equal(res.trk_y, res.tl_par[sd, 0]) and np.array_equal(res.trk_qpt, res.tl_par[sd, 4])
    assert np.array_equal(res.trk_chi2, res.tl_chi2[sd]) and np.array_equal(res.trk_ndf, 2 * nh[sd] - 5)
    assert np.array_equal(res.trk_sector, np.searchsorted(res.seed_offset, sd, side="right") - 1)
    assert np.all(np.diff(sd) > 0), "canonical order (sector, start row, start-hit index)"


def test_degenerate_inputs(oracle_mod, gen_mod):
    rx = gen_mod.row_x().astype(np.float32)
    g = oracle_mod.Geometry(36, rx, gen_mod.TAN_HALF_ANGLE, 0.06, 0.06, 0.5)
    z = np.zeros(0, np.float32)
    res = oracle_mod.track_event(g, np.zeros(37, np.int32), z, z, np.zeros(0, np.int32))
    assert res.n_tracks == 0 and res.n_seeds == 0
    # one hit, two hits in adjacent rows: no triplet, no link, no track
    so = np.zeros(37, np.int32); so[4:] = 2
    res = oracle_mod.track_event(g, so, np.array([0, 0.1], np.float32), np.array([10, 10.1], np.float32),
                                 np.array([5, 6], np.int32))
    assert res.n_tracks == 0 and np.all(res.link_up == -1)
    with pytest.raises(ValueError):
        oracle_mod.track_event(g, so, np.zeros(2, np.float32), np.zeros(2, np.float32), np.array([5, 159], np.int32))


THRESHOLDS = {"single_sector": 0.95, "pp": 0.95, "semicentral": 0.95, "central": 0.90}


@pytest.mark.parametrize("name", ["single_sector", "pp", "semicentral", "central"])
@pytest.mark.parametrize("precision", ["double", "float"])
def test_efficiency_and_fake_rate(event_and_oracle, name, precision):
    """Stated thresholds: efficiency for primaries with pT > 0.2 GeV and >= 30 clusters in a
    sector, matched by >= 90 % label purity: >= 95 % (configs 1-3), >= 90 % (config 4); fake rate <= 2 %."""
    if name == "central" and precision == "double":
        pytest.skip("central is checked in the float mode only (CPU time)")
    ev, res = event_and_oracle(name, precision)
    e = efficiency(ev, res.trk_sector, res.trk_first_hit, res.trk_n_hits, res.hit_idx)
    assert e["n_reconstructable"] >= 40
    assert e["efficiency"] >= THRESHOLDS[name], e
    assert e["fake_rate"] <= 0.02, e


def test_float_and_double_modes_agree_on_almost_everything(event_and_oracle):
    """The float32 mode is the same algorithm: on config 3 it flips only decisions with tiny margins."""
    ev, a = event_and_oracle("semicentral", "double")
    _, b = event_and_oracle("semicentral", "float")
    d = a.link_up != b.link_up
    assert d.sum() <= 20 and np.all(a.nf_margin[d] < 1e-4)
    if a.n_seeds == b.n_seeds:
        dt = (a.tl_table != b.tl_table).any(axis=1)
        assert dt.sum() <= 0.002 * a.n_seeds
        same = ~dt
        rel = np.abs(a.tl_par[same] - b.tl_par[same]) / np.maximum(1, np.abs(a.tl_par[same]))
        assert rel.max() < 5e-3
