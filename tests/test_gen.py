"""Generator self-checks (SURVEY.md 8(c).5 "Generator" pin): closed forms of the helix, acceptance, recipes."""
import math

import numpy as np

from paper_1712_09416_b200 import gen

K = 0.00299792458


def _global_xy(ev):
    sector = np.repeat(np.arange(ev.n_sectors), np.diff(ev.sector_offset))
    alpha = gen.sector_alpha(36)[sector % 18] if ev.n_sectors == 36 else np.full(ev.n_clusters, math.radians(10.0))
    x = ev.x.astype(np.float64); y = ev.y.astype(np.float64)
    return x * np.cos(alpha) - y * np.sin(alpha), x * np.sin(alpha) + y * np.cos(alpha), sector


def test_row_table():
    rx = gen.row_x()
    assert rx.shape == (159,)
    assert abs(rx[0] - 85.225) < 1e-12 and abs(rx[62] - (85.225 + 0.75 * 62)) < 1e-12
    assert abs(rx[63] - 135.1) < 1e-12 and abs(rx[127] - 199.35) < 1e-12 and abs(rx[158] - 245.85) < 1e-9
    assert np.all(np.diff(rx) > 0)


def test_unsmeared_hits_lie_on_their_helix():
    r = gen.Recipe("clean", n_primaries=40, frac_secondaries=0.5, sigma=0.0, inefficiency=0.0, noise_frac=0.0,
                   loopers=True, config_id=9)
    ev = gen.generate(r)
    assert ev.n_clusters > 3000 and np.all(ev.label >= 0)
    gx, gy, sector = _global_xy(ev)
    T = ev.tracks[ev.label]
    pt, q, eta, phi, vx, vy, vz = (T[:, i] for i in range(7))
    R = pt / (K * ev.bz)
    h = -q
    cx = vx - h * R * np.sin(phi); cy = vy + h * R * np.cos(phi)
    # on the circle (float32 storage of y at |y| < 45 cm: 4e-6 cm)
    rr = np.hypot(gx - cx, gy - cy)
    assert np.max(np.abs(rr - R) / R) < 1e-6
    # z = vz + t * R * turning angle, angle measured in the direction of motion
    psi0 = np.arctan2(vy - cy, vx - cx); psi = np.arctan2(gy - cy, gx - cx)
    th = np.mod(h * (psi - psi0), 2 * np.pi)
    t = np.sinh(eta)
    dz = ev.z - vz
    turns = np.round((dz / (t * R) - th) / (2 * np.pi))
    assert np.all(turns >= 0) and np.all(turns <= 2)
    assert np.max(np.abs(vz + t * R * (th + 2 * np.pi * turns) - ev.z)) < 2e-4
    # acceptance: inside the wedge, inside the drift length, on the right side
    assert np.all(np.abs(ev.y) <= ev.x * gen.TAN_HALF_ANGLE * (1 + 1e-6))
    assert np.all(np.abs(ev.z) <= gen.Z_MAX + 1e-3)
    assert np.all((ev.z < 0) == (sector >= 18))
    assert np.all(np.hypot(gx, gy) <= gen.R_MAX + 2.0)


def test_every_crossed_row_has_a_hit_for_stiff_primaries():
    r = gen.Recipe("stiff", n_sectors=1, n_primaries=20, pt_mode=0, pt_a=2.0, pt_b=5.0, sigma=0.0, inefficiency=0.0,
                   noise_frac=0.0, config_id=8)
    ev = gen.generate(r)
    for t in range(20):
        rows = np.sort(ev.row[ev.label == t])
        assert rows.size >= 20 and rows[0] == 0      # may leave the wedge early, never skips a row
        assert np.all(np.diff(rows) == 1), "an outgoing stiff track crosses consecutive rows once each"


def test_recipes_sizes_and_determinism():
    a = gen.generate("single_sector"); b = gen.generate("single_sector")
    assert a.n_clusters == b.n_clusters and np.array_equal(a.y, b.y) and np.array_equal(a.row, b.row)
    assert 6000 < a.n_clusters < 9000          # BASELINE.json:7 "~8k clusters"
    assert a.seed == 1000
    c = gen.generate("single_sector", event=1)
    assert c.seed == 1001 and not np.array_equal(a.y[:100], c.y[:100])
    pp = gen.generate("pp")
    assert 7000 < pp.n_clusters < 13000        # BASELINE.json:8 "~10k"
    assert pp.sector_offset.shape == (37,) and pp.sector_offset[-1] == pp.n_clusters
    noise = (pp.label < 0).mean()
    assert 0.03 < noise < 0.06
    sc = gen.generate("semicentral")
    assert 300_000 < sc.n_clusters < 420_000   # BASELINE.json:9 "~350k"
    assert sc.tracks.shape[0] == 2300 and int(sc.tracks[:, 7].sum()) == 2000


def test_smearing_and_inefficiency_statistics():
    base = dict(n_sectors=1, n_primaries=200, pt_mode=0, pt_a=1.0, pt_b=5.0, noise_frac=0.0, config_id=7)
    clean = gen.generate(gen.Recipe("c", sigma=0.0, inefficiency=0.0, shuffle=False, **base))
    noisy = gen.generate(gen.Recipe("n", sigma=0.06, inefficiency=0.02, shuffle=False, **base))
    loss = 1.0 - noisy.n_clusters / clean.n_clusters
    assert 0.012 < loss < 0.028
    # the smearing stream is independent of acceptance: match hits by (label, row)
    kc = clean.label.astype(np.int64) * 1000 + clean.row
    kn = noisy.label.astype(np.int64) * 1000 + noisy.row
    idx = {k: i for i, k in enumerate(kc)}
    sel = np.array([idx[k] for k in kn])
    dy = noisy.y - clean.y[sel]; dz = noisy.z - clean.z[sel]
    assert abs(dy.std() - 0.06) < 0.002 and abs(dz.std() - 0.06) < 0.002
    assert abs(dy.mean()) < 0.002 and abs(dz.mean()) < 0.002
