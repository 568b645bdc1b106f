"""Pins of the oracle's O9 (cross-sector merge of track segments).

* against the generator's truth: a generated particle that crosses a sector border and is reconstructed on both
  sides must come out linked (efficiency per crossing), and linked segments must belong to the same particle,
* structure: links are mutual and one-to-one, join neighbouring sectors of the same side, lower segment first,
* geometry, independently: for every link the first segment's outer state, turned into the second's frame and moved
  along the EXACT helix (closed form with asin, written here in double), lands on the second segment's parameters
  within the tolerances.
"""
import math

import numpy as np
import pytest

from test_oracle_kf import K


def _run(oracle, gen, name, event=0, precision="float", **kw):
    ev = gen.generate(name, event)
    g = oracle.Geometry(ev.n_sectors, gen.row_x().astype(np.float32), gen.TAN_HALF_ANGLE, ev.sigma, ev.sigma, ev.bz)
    p = oracle.default_params()
    p.refit = 1
    p.merge = 1
    for k, v in kw.items():
        setattr(p, k, v)
    return ev, p, oracle.track_event(g, ev.sector_offset, ev.y, ev.z, ev.row, params=p, precision=precision)


def _labels(ev, r):
    lab = np.full(r.n_tracks, -1)
    pur = np.zeros(r.n_tracks)
    for i in range(r.n_tracks):
        h = r.hit_idx[r.trk_first_hit[i]:r.trk_first_hit[i] + r.trk_n_hits[i]]
        v, c = np.unique(ev.label[h], return_counts=True)
        j = c.argmax()
        lab[i], pur[i] = v[j], c[j] / len(h)
    return lab, pur


@pytest.mark.parametrize("name,min_eff", [("pp", 0.98), ("semicentral", 0.98), ("central", 0.98)])
def test_merge_links_the_segments_of_one_particle(oracle_mod, gen_mod, name, min_eff):
    ev, p, r = _run(oracle_mod, gen_mod, name)
    lab, pur = _labels(ev, r)
    good = (pur >= 0.9) & (lab >= 0)
    half = ev.n_sectors // 2
    sec = r.trk_sector
    merged = {(a, int(r.trk_next[a])) for a in range(r.n_tracks) if r.trk_next[a] >= 0}
    by = {}
    for i in np.nonzero(good)[0]:
        by.setdefault(lab[i], []).append(i)
    crossings = {}
    for idx in by.values():
        for a in idx:
            for b in idx:
                if a == b or sec[a] // half != sec[b] // half:
                    continue
                if (sec[b] % half - sec[a] % half) % half not in (1, half - 1):
                    continue
                if 1 <= r.trk_first_row[b] - r.trk_row_out[a] <= 1 + p.merge_max_gap:
                    crossings.setdefault((lab[a], sec[a], sec[b]), []).append((a, b) in merged)
    assert len(crossings) >= (40 if name == "pp" else 1000)
    eff = np.mean([any(v) for v in crossings.values()])
    fake = np.mean([lab[a] != lab[b] or not good[a] or not good[b] for a, b in merged])
    assert eff >= min_eff, eff
    assert fake <= 0.005, fake


def test_merge_structure(oracle_mod, gen_mod):
    ev, p, r = _run(oracle_mod, gen_mod, "semicentral")
    half = ev.n_sectors // 2
    nx, pv = r.trk_next, r.trk_prev
    a = np.nonzero(nx >= 0)[0]
    assert a.size > 1000
    assert np.array_equal(pv[nx[a]], a)                              # mutual
    assert np.unique(nx[a]).size == a.size                           # one-to-one
    b = np.nonzero(pv >= 0)[0]
    assert np.array_equal(nx[pv[b]], b)
    sa, sb = r.trk_sector[a], r.trk_sector[nx[a]]
    assert np.all(sa // half == sb // half)
    assert np.all(np.isin((sb % half - sa % half) % half, (1, half - 1)))
    gap = r.trk_first_row[nx[a]] - r.trk_row_out[a]
    assert np.all((gap >= 1) & (gap <= 1 + p.merge_max_gap))
    # switched off: no links, tracks unchanged
    ev2, p2, r2 = _run(oracle_mod, gen_mod, "semicentral", merge=0)
    assert np.all(r2.trk_next == -1) and np.all(r2.trk_prev == -1)
    assert np.array_equal(r2.trk_qpt, r.trk_qpt) and np.array_equal(r2.hit_idx, r.hit_idx)
    # the merge needs the refit's outer states
    ev3, p3, r3 = _run(oracle_mod, gen_mod, "pp", refit=0)
    assert np.all(r3.trk_next == -1)


def _exact_move(x, y, z, s, t, q, x1, bz):
    """Closed-form helix from x to x1 (state y, z, sin phi, tg lambda, q/pT), double."""
    kap = -K * bz * q
    s1 = s + kap * (x1 - x)
    c, c1 = math.sqrt(1 - s * s), math.sqrt(1 - s1 * s1)
    dy = (x1 - x) * (s + s1) / (c + c1)
    if abs(kap) < 1e-12:
        dS = math.hypot(x1 - x, dy)
    else:
        dS = (math.asin(s1) - math.asin(s)) / kap
    return y + dy, z + t * dS, s1


def test_merge_links_agree_with_exact_helix_geometry(oracle_mod, gen_mod):
    ev, p, r = _run(oracle_mod, gen_mod, "semicentral", precision="double")
    half = ev.n_sectors // 2
    step = 2 * math.pi / half
    n = 0
    for a in np.nonzero(r.trk_next >= 0)[0]:
        b = int(r.trk_next[a])
        xo, yo, zo, so, to, qo = r.trk_out[a]
        dk = (r.trk_sector[b] % half - r.trk_sector[a] % half) % half
        ang = -step if dk == 1 else step                      # alpha_A - alpha_B
        phi = math.asin(so) + ang
        x1 = xo * math.cos(ang) - yo * math.sin(ang)
        y1 = xo * math.sin(ang) + yo * math.cos(ang)
        y2, z2, s2 = _exact_move(x1, y1, zo, math.sin(phi), to, qo, r.trk_x[b], ev.bz)
        assert abs(y2 - r.trk_y[b]) <= p.merge_dy * (1 + 1e-6) and abs(z2 - r.trk_z[b]) <= p.merge_dz * (1 + 1e-6)
        assert abs(s2 - r.trk_sinphi[b]) <= p.merge_ds * (1 + 1e-6) and abs(to - r.trk_tgl[b]) <= p.merge_dt * (1 + 1e-6)
        n += 1
    assert n > 1000


def test_global_tracks_are_the_chains_of_links(oracle_mod, gen_mod):
    """trk_global names every segment's chain by its first segment: heads have no predecessor, a link never joins
    two chains, chains grow outwards, and (truth) the segments of a chain belong to one particle."""
    ev, p, r = _run(oracle_mod, gen_mod, "semicentral")
    g, nx, pv = r.trk_global, r.trk_next, r.trk_prev
    T = r.n_tracks
    assert np.all(pv[g] == -1) and np.all(g[g] == g)
    assert np.array_equal(g[pv >= 0], g[pv[pv >= 0]])            # a segment and its predecessor: same chain
    assert np.all(g[pv < 0] == np.nonzero(pv < 0)[0])            # heads name themselves
    a = np.nonzero(nx >= 0)[0]
    assert np.all(r.trk_first_row[nx[a]] > r.trk_row_out[a])     # outwards
    sizes = np.bincount(g, minlength=T)
    assert sizes.max() >= 2 and sizes.max() <= ev.n_sectors // 2
    lab, pur = _labels(ev, r)
    multi = np.nonzero(sizes >= 2)[0]
    same = [np.unique(lab[g == h]).size == 1 for h in multi[:400]]
    assert np.mean(same) > 0.995
    # merge off: every track is its own global track
    ev2, p2, r2 = _run(oracle_mod, gen_mod, "pp", merge=0)
    assert np.array_equal(r2.trk_global, np.arange(r2.n_tracks))
