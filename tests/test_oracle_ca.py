"""Pins of the oracle's Cellular-Automaton stage (O2 neighbour finder, O3 cleaner, O4 start hits).

SURVEY.md 8(c).5: brute force over all (d, h, u) triplets on tiny sectors gives identical links; the deviation is
invariant under the mirror y -> -y; cleaned links are mutual and cleaning is idempotent; start hits are the lower
ends of maximal chains.  The brute force below is written from the definition with numpy outer
products; it shares nothing with oracle/tpc_oracle.cpp.
"""
import numpy as np
import pytest

from conftest import make_geometry


def brute_force_links(ev, row_x, p, dtype):
    """All-triplets search, straight from the definition.  Returns (link_up, link_dn) in event indices."""
    f = dtype
    N = ev.n_clusters
    up = np.full(N, -1, np.int32); dn = np.full(N, -1, np.int32)
    X = row_x.astype(np.float32).astype(f)
    y = ev.y.astype(f); z = ev.z.astype(f)
    D = p.link_step
    Ty, Tz, w0, Dmax = f(p.nf_slope_y), f(p.nf_slope_z), f(p.nf_w0), f(p.nf_dmax)
    for s in range(ev.n_sectors):
        b, e = ev.sector_offset[s], ev.sector_offset[s + 1]
        idx = np.arange(b, e)
        rows = ev.row[b:e]
        for r in range(D, len(X) - D):
            H = idx[rows == r]; U = idx[rows == r + D]; Dn = idx[rows == r - D]
            if H.size == 0 or U.size == 0 or Dn.size == 0:
                continue
            x0, x1, x2 = X[r], X[r + D], X[r - D]
            a = (x0 - x2) / (x1 - x2)
            wyu = Ty * abs(x1 - x0) + w0; wzu = Tz * abs(x1 - x0) + w0
            wyd = Ty * abs(x2 - x0) + w0; wzd = Tz * abs(x2 - x0) + w0
            for h in H:
                inu = (np.abs(y[U] - y[h]) <= wyu) & (np.abs(z[U] - z[h]) <= wzu)
                ind = (np.abs(y[Dn] - y[h]) <= wyd) & (np.abs(z[Dn] - z[h]) <= wzd)
                if not inu.any() or not ind.any():
                    continue
                yh = y[Dn][None, :] + a * (y[U][:, None] - y[Dn][None, :])
                zh = z[Dn][None, :] + a * (z[U][:, None] - z[Dn][None, :])
                dy = y[h] - yh; dz = z[h] - zh
                dev = dy * dy + dz * dz
                dev = np.where(inu[:, None] & ind[None, :], dev, f(np.inf))
                k = int(np.argmin(dev))              # first minimum in (u, d) row-major order = lowest u then d
                iu, idn = divmod(k, Dn.size)
                if dev[iu, idn] <= Dmax:
                    up[h] = U[iu]; dn[h] = Dn[idn]
    return up, dn


@pytest.mark.parametrize("step", [1, 2])
@pytest.mark.parametrize("precision,dtype", [("double", np.float64), ("float", np.float32)])
def test_links_equal_brute_force(oracle_mod, gen_mod, step, precision, dtype):
    p = oracle_mod.default_params()
    p.link_step = step
    for seed, ntr, noise in ((7, 6, 0.5), (8, 12, 1.0), (9, 25, 0.3)):
        ev = gen_mod.tiny_sector(n_tracks=ntr, seed=seed, noise_frac=noise)
        res = oracle_mod.track_event(make_geometry(oracle_mod, gen_mod, ev), ev.sector_offset, ev.y, ev.z, ev.row,
                                     params=p, precision=precision, stop_after=4)
        up, dn = brute_force_links(ev, gen_mod.row_x(), p, dtype)
        assert (up >= 0).sum() > 0.5 * (ev.label >= 0).sum() * (0.9 if step == 1 else 0.8)
        assert np.array_equal(res.link_up, up)
        assert np.array_equal(res.link_dn, dn)


def test_links_on_dense_ambiguous_rows_equal_brute_force(oracle_mod, gen_mod):
    """Many candidates per window: a pure-noise sector squeezed into few rows (<= 40 hits per row)."""
    rng = np.random.default_rng(5)
    n_rows_used, per_row = 7, 40
    rx = gen_mod.row_x()
    row = np.repeat(np.arange(50, 50 + n_rows_used), per_row).astype(np.int32)
    y = rng.uniform(-3, 3, row.size).astype(np.float32)
    z = rng.uniform(100, 106, row.size).astype(np.float32)
    perm = rng.permutation(row.size)
    ev = gen_mod.Event(1, np.array([0, row.size], np.int32), rx[row[perm]].astype(np.float32), y[perm], z[perm],
                       row[perm], np.full(row.size, -1, np.int32), np.zeros((0, 8)))
    p = oracle_mod.default_params()
    p.nf_dmax = 2.0
    for precision, dtype in (("double", np.float64), ("float", np.float32)):
        res = oracle_mod.track_event(make_geometry(oracle_mod, gen_mod, ev), ev.sector_offset, ev.y, ev.z, ev.row,
                                     params=p, precision=precision, stop_after=4)
        up, dn = brute_force_links(ev, rx, p, dtype)
        assert (up >= 0).sum() > 100
        assert np.array_equal(res.link_up, up) and np.array_equal(res.link_dn, dn)


def test_coincident_hits_tie_goes_to_lowest_index(oracle_mod, gen_mod):
    """S22: identical (y, z) in a row are legal; the lowest original index wins every tie."""
    rx = gen_mod.row_x()
    row = np.array([10, 11, 11, 12, 12, 12], np.int32)
    y = np.array([0.0, 0.1, 0.1, 0.2, 0.2, 0.2], np.float32)
    z = np.array([50.0, 50.5, 50.5, 51.0, 51.0, 51.0], np.float32)
    ev = gen_mod.Event(1, np.array([0, 6], np.int32), rx[row].astype(np.float32), y, z, row,
                       np.zeros(6, np.int32), np.zeros((1, 8)))
    res = oracle_mod.track_event(make_geometry(oracle_mod, gen_mod, ev), ev.sector_offset, y, z, row, stop_after=4)
    assert res.link_up[1] == 3 and res.link_dn[1] == 0 and res.link_up[2] == 3 and res.link_dn[2] == 0
    # hit 3 (lowest index of the triple) is linked back by... nobody twice: cleaned links stay mutual
    assert res.clink_up[1] == -1 or res.clink_dn[res.clink_up[1]] == 1


@pytest.mark.parametrize("precision", ["double", "float"])
def test_deviation_equal_to_d_max_is_accepted(oracle_mod, gen_mod, precision):
    """"If D_best <= D_max" -- the bound itself is accepted.  Three hits on rows 10, 11, 12 at
    z = 50: the outer two at y = 0, the middle one at y0.  The interpolated point is (0, 50) whatever the row pitch, so
    D = y0^2 exactly: y0 = 0.5 gives D = 0.25 = nf_dmax (exact in float32 and double) -> the link is made; the next
    float32 above 0.5 gives D > 0.25 -> no link.  Kills the mutant `D_best < D_max` of oracle/tpc_oracle.cpp
    `neighbours`."""
    rx = gen_mod.row_x()
    p = oracle_mod.default_params()
    assert p.nf_dmax == 0.25 and p.nf_slope_y * (rx[11] - rx[10]) + p.nf_w0 > 0.6     # the windows do not decide here
    row = np.array([10, 11, 12], np.int32)
    z = np.full(3, 50.0, np.float32)
    for y0, linked in ((np.float32(0.5), True), (np.nextafter(np.float32(0.5), np.float32(1)), False),
                       (np.float32(-0.5), True), (np.nextafter(np.float32(-0.5), np.float32(-1)), False)):
        y = np.array([0.0, y0, 0.0], np.float32)
        ev = gen_mod.Event(1, np.array([0, 3], np.int32), rx[row].astype(np.float32), y, z, row, np.zeros(3, np.int32),
                           np.zeros((1, 8)))
        res = oracle_mod.track_event(make_geometry(oracle_mod, gen_mod, ev), ev.sector_offset, y, z, row,
                                     precision=precision, stop_after=4)
        assert (res.link_up[1], res.link_dn[1]) == ((2, 0) if linked else (-1, -1)), (float(y0), precision)
        assert res.link_up[0] == res.link_up[2] == -1


def test_mirror_symmetry(oracle_mod, gen_mod):
    """D(h; u, d) is invariant under y -> -y, so the links of the mirrored sector are the same."""
    ev = gen_mod.tiny_sector(n_tracks=20, seed=11, noise_frac=0.5)
    g = make_geometry(oracle_mod, gen_mod, ev)
    a = oracle_mod.track_event(g, ev.sector_offset, ev.y, ev.z, ev.row, stop_after=4)
    b = oracle_mod.track_event(g, ev.sector_offset, -ev.y, ev.z, ev.row, stop_after=4)
    for k in ("link_up", "link_dn", "clink_up", "clink_dn", "start_hit"):
        assert np.array_equal(a[k], b[k])


@pytest.mark.parametrize("name", ["single_sector", "pp", "semicentral"])
def test_cleaner_and_start_hit_invariants(event_and_oracle, name):
    ev, res = event_and_oracle(name, "float")
    N = ev.n_clusters
    lu, ld, cu, cd = res.link_up, res.link_dn, res.clink_up, res.clink_dn
    # links come in pairs before cleaning and point to the adjacent rows of the same sector
    assert np.array_equal(lu >= 0, ld >= 0)
    h = np.nonzero(lu >= 0)[0]
    assert np.all(ev.row[lu[h]] == ev.row[h] + 1) and np.all(ev.row[ld[h]] == ev.row[h] - 1)
    sector = np.repeat(np.arange(ev.n_sectors), np.diff(ev.sector_offset))
    assert np.all(sector[lu[h]] == sector[h]) and np.all(sector[ld[h]] == sector[h])
    # O3 from its definition, in numpy
    exp_cu = np.where((lu >= 0) & (ld[np.maximum(lu, 0)] == np.arange(N)), lu, -1)
    exp_cd = np.where((ld >= 0) & (lu[np.maximum(ld, 0)] == np.arange(N)), ld, -1)
    assert np.array_equal(cu, exp_cu) and np.array_equal(cd, exp_cd)
    # mutual
    u = np.nonzero(cu >= 0)[0]; d = np.nonzero(cd >= 0)[0]
    assert np.all(cd[cu[u]] == u) and np.all(cu[cd[d]] == d)
    # idempotent: cleaning the cleaned links changes nothing
    cu2 = np.where((cu >= 0) & (cd[np.maximum(cu, 0)] == np.arange(N)), cu, -1)
    cd2 = np.where((cd >= 0) & (cu[np.maximum(cd, 0)] == np.arange(N)), cd, -1)
    assert np.array_equal(cu2, cu) and np.array_equal(cd2, cd)
    # O4: start hits = hits with an up link and no down link, in (sector, row, index) order
    flag = (cu >= 0) & (cd < 0)
    order = np.lexsort((np.arange(N), ev.row, sector))
    exp = order[flag[order]]
    assert np.array_equal(res.start_hit, exp)
    assert np.array_equal(res.seed_offset, np.concatenate([[0], np.cumsum(np.bincount(sector[exp], minlength=ev.n_sectors))]))
    # number of start hits = number of maximal chains (walk every chain down from its top end)
    tops = np.nonzero((cd >= 0) & (cu < 0))[0]
    assert tops.size == exp.size
    seen = set()
    for t in tops:
        k = t
        while cd[k] >= 0:
            k = cd[k]
        seen.add(int(k))
    assert seen == set(int(v) for v in exp)
