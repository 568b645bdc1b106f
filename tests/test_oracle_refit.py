"""Pins of the oracle's O8 (refit of a selected track over its final hit list).

* against the generated helix (noise-free hits: the parameters are the helix's),
* against the textbook least-squares line (Bz -> 0),
* against a step-by-step composition, written here, of the two primitives that are pinned on their own in
  test_oracle_kf.py (transport against the closed-form helix, update against the textbook Kalman update): this
  checks the refit's orchestration -- first hit, direction from the first two hits, transport to EVERY row,
  measurements only on the list's rows, fresh down pass from the top hit, reference row, ndf,
* statistically with noise (chi2/ndf, curvature resolution against Gluckstern's formula).
"""
import math

import numpy as np
import pytest

from test_oracle_kf import BZ, K, _single_track_events, truth_state


def _geom(oracle, gen, sigma=0.06, bz=BZ, n_sectors=1):
    return oracle.Geometry(n_sectors, gen.row_x().astype(np.float32), gen.TAN_HALF_ANGLE, sigma, sigma, bz)


def _params(oracle, refit):
    p = oracle.default_params()
    p.refit = refit
    return p


def test_refit_off_is_the_default_and_changes_nothing(oracle_mod, gen_mod):
    ev = gen_mod.generate("single_sector")
    g = _geom(oracle_mod, gen_mod, ev.sigma, ev.bz)
    a = oracle_mod.track_event(g, ev.sector_offset, ev.y, ev.z, ev.row, precision="float")
    b = oracle_mod.track_event(g, ev.sector_offset, ev.y, ev.z, ev.row, precision="float", params=_params(oracle_mod, 0))
    c = oracle_mod.track_event(g, ev.sector_offset, ev.y, ev.z, ev.row, precision="float", params=_params(oracle_mod, 1))
    assert oracle_mod.default_params().refit == 0
    for k in ("hit_idx", "trk_n_hits", "trk_first_hit", "trk_sector"):
        assert np.array_equal(a[k], b[k]) and np.array_equal(a[k], c[k])      # the refit never touches hit lists
    for k in ("trk_y", "trk_qpt", "trk_chi2"):
        assert np.array_equal(a[k], b[k])
    assert not np.array_equal(a["trk_qpt"], c["trk_qpt"])


def test_refit_recovers_noise_free_helix(oracle_mod, gen_mod):
    used = 0
    for ev in _single_track_events(gen_mod, 16, sigma=0.0, pt_a=0.25, pt_b=3.0):
        if ev.n_clusters < 60:
            continue
        used += 1
        g = _geom(oracle_mod, gen_mod)
        res = oracle_mod.track_event(g, ev.sector_offset, ev.y, ev.z, ev.row, precision="double",
                                     params=_params(oracle_mod, 1))
        assert res.n_tracks == 1 and res.trk_n_hits[0] == ev.n_clusters
        assert res.trk_ndf[0] == 2 * ev.n_clusters - 5
        assert res.trk_x[0] == np.float32(gen_mod.row_x()[ev.row.min()])        # reference = lowest hit's row
        tr = truth_state(ev.tracks[0], res.trk_x[0])
        fit = np.array([res.trk_y[0], res.trk_z[0], res.trk_sinphi[0], res.trk_tgl[0], res.trk_qpt[0]])
        assert np.all(np.abs(fit - tr) < np.array([2e-5, 4e-5, 2e-6, 2e-6, 2e-4])), (fit, tr)
        assert res.trk_chi2[0] < 1e-4
    assert used >= 8


def test_refit_straight_line_limit_equals_least_squares(oracle_mod, gen_mod):
    bz = 1e-7
    for ev in _single_track_events(gen_mod, 10, sigma=0.06, pt_a=1.0, pt_b=2.0, bz=bz):
        g = _geom(oracle_mod, gen_mod, 0.06, bz)
        res = oracle_mod.track_event(g, ev.sector_offset, ev.y, ev.z, ev.row, precision="double",
                                     params=_params(oracle_mod, 1))
        assert res.n_tracks == 1 and res.trk_n_hits[0] == ev.n_clusters
        x = ev.x.astype(np.float64); xr = res.trk_x[0]
        A = np.stack([np.ones_like(x), x - xr], axis=1)
        (y0, ty), *_ = np.linalg.lstsq(A, ev.y.astype(np.float64), rcond=None)
        (z0, tz), *_ = np.linalg.lstsq(A, ev.z.astype(np.float64), rcond=None)
        s_ls = ty / math.sqrt(1 + ty * ty)
        t_ls = tz * math.sqrt(1 - s_ls * s_ls)
        assert abs(res.trk_y[0] - y0) < 2e-4 and abs(res.trk_z[0] - z0) < 2e-4
        assert abs(res.trk_sinphi[0] - s_ls) < 5e-6 and abs(res.trk_tgl[0] - t_ls) < 1e-5


outer_of = {}   # filled by _compose_refit: what the up pass of the last composed track handed over


def _compose_refit(oracle, g, rx, ev, hits):
    """O8 written out with the pinned primitives: returns (params[5], chi2, n_fit, ref_row)."""
    p = oracle.default_params()
    sy, sz = float(np.float32(g.sigma_y)), float(np.float32(g.sigma_z))     # the geometry carries float32
    prior = np.diag([sy * sy, sz * sz, p.var_s, p.var_t, p.var_q]).astype(np.float64)
    y, z, row = ev.y.astype(np.float64), ev.z.astype(np.float64), ev.row
    rows = [int(row[h]) for h in hits]
    h0, h1 = hits[0], hits[1]
    dx = float(rx[rows[1]]) - float(rx[rows[0]])
    dy, dz = y[h1] - y[h0], z[h1] - z[h0]
    dl = math.sqrt(dx * dx + dy * dy)
    st = np.array([y[h0], z[h0], dy / dl, dz / dl, 0.0]); cv = prior.copy(); chi2 = 0.0
    snap = (st.copy(), chi2, 1)
    outer_of.clear()
    on_row = {r: h for r, h in zip(rows, hits)}
    k_top_row = rows[0]
    xc = float(rx[rows[0]])
    for r in range(rows[0] + 1, rows[-1] + 1):
        ok, st, cv = oracle.transport(g, xc, float(rx[r]), st, cv)
        if not ok:
            break
        xc = float(rx[r])
        if r in on_row:
            st, cv, chi2 = oracle.update(g, y[on_row[r]], z[on_row[r]], st, cv, chi2)
            snap = (st.copy(), chi2, 0); k_top_row = r
    # the refit's OUTER state: the up pass right after its last update, not where the pass ended
    outer_of.update(state=snap[0].copy(), row=k_top_row, running=st.copy(), ended_early=k_top_row < rows[-1])
    ht = on_row[k_top_row]
    st = np.array([y[ht], z[ht], snap[0][2], snap[0][3], snap[0][4]]); cv = prior.copy(); chi2 = 0.0
    out = (st.copy(), 0.0, 1, k_top_row)
    n = 1
    xc = float(rx[k_top_row])
    for r in range(k_top_row - 1, rows[0] - 1, -1):
        ok, st, cv = oracle.transport(g, xc, float(rx[r]), st, cv)
        if not ok:
            break
        xc = float(rx[r])
        if r in on_row:
            st, cv, chi2 = oracle.update(g, y[on_row[r]], z[on_row[r]], st, cv, chi2)
            n += 1
            out = (st.copy(), chi2, n, r)
    return out


def test_refit_equals_composition_of_pinned_primitives(oracle_mod, gen_mod):
    """Tracks of a busy single sector (holes, noise, hits lost to other tracks in the selection)."""
    ev = gen_mod.generate("single_sector")
    g = _geom(oracle_mod, gen_mod, ev.sigma, ev.bz)
    rx = gen_mod.row_x().astype(np.float32)
    res = oracle_mod.track_event(g, ev.sector_offset, ev.y, ev.z, ev.row, precision="double",
                                 params=_params(oracle_mod, 1))
    base = oracle_mod.track_event(g, ev.sector_offset, ev.y, ev.z, ev.row, precision="double")
    assert res.n_tracks > 30
    holes = 0
    for i in range(res.n_tracks):
        hits = [int(h) for h in res.hit_idx[res.trk_first_hit[i]:res.trk_first_hit[i] + res.trk_n_hits[i]]]
        rows = ev.row[hits]
        assert np.all(np.diff(rows) > 0)
        holes += int(rows[-1] - rows[0] + 1 - len(rows))
        st, chi2, n, ref_row = _compose_refit(oracle_mod, g, rx, ev, hits)
        fit = np.array([res.trk_y[i], res.trk_z[i], res.trk_sinphi[i], res.trk_tgl[i], res.trk_qpt[i]])
        assert np.allclose(fit, st, rtol=1e-12, atol=1e-14), (i, fit, st)
        assert abs(res.trk_chi2[i] - chi2) <= 1e-12 * max(1.0, chi2)
        assert res.trk_ndf[i] == 2 * n - 5 and res.trk_first_row[i] == ref_row
        assert res.trk_x[i] == rx[ref_row]
        assert res.trk_row_out[i] == outer_of["row"] == rows[-1] and res.trk_out[i, 0] == rx[outer_of["row"]]
        assert np.allclose(res.trk_out[i, 1:], outer_of["state"], rtol=1e-12, atol=1e-14)
    assert holes > 20                      # rows without a measurement inside the tracks were exercised
    assert np.any(base.trk_n_hits != (base.trk_ndf + 5) // 2)   # the selection did take hits from some tracklets


def test_refit_outer_state_is_the_last_snapshot_when_the_up_pass_ends_early(oracle_mod, gen_mod):
    """pT 0.08-0.16 GeV curlers: the refit's up pass reaches |sin phi| = s_max before the track's last hit, some rows
    AFTER its last update (rows without a hit were crossed in between).  The outer state (trk_out, trk_row_out, the
    input of the cross-sector match O9) is then the snapshot taken at the last update, at that hit's row -- not the
    running fit at the row where the pass ended.  Composition of the pinned transport / update primitives, as in the
    test above.  Kills the mutant of oracle/tpc_oracle.cpp `refit` that copies the running fit `f` into `out`."""
    r = gen_mod.Recipe("curlers", n_sectors=36, n_primaries=1500, pt_mode=0, pt_a=0.08, pt_b=0.16, sigma=0.06,
                       noise_frac=0.05, config_id=61)
    full = gen_mod.generate(r)
    # 30 % of the clusters are dropped at random (seeded): the tracks get holes, so that a pass which ends between two
    # hits has often crossed rows since its last update
    keep = np.random.default_rng(5).random(full.row.size) < 0.7
    so = np.concatenate([[0], np.cumsum([int(keep[a:b].sum()) for a, b in zip(full.sector_offset[:-1],
                                                                               full.sector_offset[1:])])])
    ev = gen_mod.Event(36, so.astype(np.int32), full.x[keep], full.y[keep], full.z[keep], full.row[keep],
                       full.label[keep], full.tracks, sigma=full.sigma)
    g = _geom(oracle_mod, gen_mod, ev.sigma, ev.bz, n_sectors=36)
    rx = gen_mod.row_x().astype(np.float32)
    res = oracle_mod.track_event(g, ev.sector_offset, ev.y, ev.z, ev.row, precision="double",
                                 params=_params(oracle_mod, 1))
    early = moved = 0
    last_row = np.array([ev.row[res.hit_idx[res.trk_first_hit[i] + res.trk_n_hits[i] - 1]] for i in range(res.n_tracks)])
    for i in sorted(set(range(150)) | set(np.nonzero(res.trk_row_out < last_row)[0].tolist())):
        hits = [int(h) for h in res.hit_idx[res.trk_first_hit[i]:res.trk_first_hit[i] + res.trk_n_hits[i]]]
        _compose_refit(oracle_mod, g, rx, ev, hits)
        assert res.trk_row_out[i] == outer_of["row"] and res.trk_out[i, 0] == rx[outer_of["row"]], i
        assert np.allclose(res.trk_out[i, 1:], outer_of["state"], rtol=1e-12, atol=1e-14), (i, res.trk_out[i], outer_of)
        early += outer_of["ended_early"]
        moved += bool(outer_of["ended_early"] and np.abs(outer_of["running"][:3] - outer_of["state"][:3]).max() > 1e-3)
    assert early >= 8 and moved >= 3, (res.n_tracks, early, moved)   # the case under test did occur


@pytest.mark.parametrize("precision", ["double", "float"])
def test_refit_chi2_and_curvature_resolution(oracle_mod, gen_mod, precision):
    sigma = 0.06
    chi2ndf, dq = [], []
    for ev in _single_track_events(gen_mod, 40, sigma=sigma, pt_a=1.0, pt_b=4.0, ineff=0.02, n_trk=10):
        g = _geom(oracle_mod, gen_mod, sigma)
        res = oracle_mod.track_event(g, ev.sector_offset, ev.y, ev.z, ev.row, precision=precision,
                                     params=_params(oracle_mod, 1))
        for i in range(res.n_tracks):
            hits = res.hit_idx[res.trk_first_hit[i]:res.trk_first_hit[i] + res.trk_n_hits[i]]
            lab = ev.label[hits]
            if res.trk_n_hits[i] < 150 or np.any(lab != lab[0]):
                continue
            assert res.trk_ndf[i] == 2 * res.trk_n_hits[i] - 5          # list and fit agree after the refit
            tr = truth_state(ev.tracks[lab[0]], res.trk_x[i])
            chi2ndf.append(res.trk_chi2[i] / res.trk_ndf[i])
            dq.append(res.trk_qpt[i] - tr[4])
    assert len(dq) > 200
    assert 0.9 < np.mean(chi2ndf) < 1.1, np.mean(chi2ndf)
    N, L = 155, 245.85 - 85.225
    gl = sigma / L ** 2 * math.sqrt(720.0 / (N + 4)) / (K * BZ)
    assert abs(np.mean(dq)) < 0.15 * gl * 3 and 0.75 * gl < np.std(dq) < 1.35 * gl, (np.mean(dq), np.std(dq), gl)
