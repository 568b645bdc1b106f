"""Truth matching of reconstructed tracks against generator labels (definitions: DESIGN.md "Efficiency").

reconstructable segment = (primary track with pT > pt_min, sector) with >= min_clusters clusters in that sector;
a reco track is *matched* to label L if >= purity of its hits carry L; found = segment with >= 1 matched track;
fake = reco track whose best label has < purity (or is noise); clone = matched tracks beyond the first per segment.
"""
from __future__ import annotations

import numpy as np


def match_tracks(ev, trk_sector, trk_first_hit, trk_n_hits, hit_idx, purity=0.9):
    """Return per-track (best_label, purity_fraction)."""
    nt = len(trk_sector)
    best = np.full(nt, -1, np.int64)
    frac = np.zeros(nt)
    lab = ev.label
    for i in range(nt):
        h = hit_idx[trk_first_hit[i]:trk_first_hit[i] + trk_n_hits[i]]
        l = lab[h]
        l = l[l >= 0]
        if l.size == 0:
            continue
        vals, cnt = np.unique(l, return_counts=True)
        k = np.argmax(cnt)
        best[i] = vals[k]
        frac[i] = cnt[k] / trk_n_hits[i]
    return best, frac


def efficiency(ev, trk_sector, trk_first_hit, trk_n_hits, hit_idx, pt_min=0.2, min_clusters=30, purity=0.9):
    n_trk = ev.tracks.shape[0]
    sector_of = np.repeat(np.arange(ev.n_sectors), np.diff(ev.sector_offset))
    sig = ev.label >= 0
    # clusters per (track, sector)
    cnt = np.zeros((n_trk, ev.n_sectors), np.int64)
    np.add.at(cnt, (ev.label[sig], sector_of[sig]), 1)
    pt = ev.tracks[:, 0]
    primary = ev.tracks[:, 7] > 0.5
    reco_able = (cnt >= min_clusters) & (primary & (pt > pt_min))[:, None]
    best, frac = match_tracks(ev, trk_sector, trk_first_hit, trk_n_hits, hit_idx, purity)
    matched = frac >= purity
    found = np.zeros_like(reco_able)
    nmatch = np.zeros((n_trk, ev.n_sectors), np.int64)
    ts = np.asarray(trk_sector)
    np.add.at(nmatch, (best[matched], ts[matched]), 1)
    found = reco_able & (nmatch > 0)
    n_reco_able = int(reco_able.sum())
    n_tracks = len(ts)
    return {
        "n_reconstructable": n_reco_able,
        "efficiency": float(found.sum()) / max(n_reco_able, 1),
        "n_tracks": n_tracks,
        "fake_rate": float((~matched).sum()) / max(n_tracks, 1),
        "clone_rate": float(np.maximum(nmatch - 1, 0).sum()) / max(n_tracks, 1),
        "best_label": best,
        "purity": frac,
    }
