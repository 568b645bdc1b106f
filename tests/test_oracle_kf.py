"""Pins of the oracle's Kalman-filter pieces (O5) against closed forms and textbook results
(SURVEY.md 8(c).5 "O5 transport" and "O5 fit").  Nothing here calls the oracle to produce its own expectation.
"""
import math

import numpy as np
import pytest

K = 0.00299792458
BZ = 0.5
KB = -K * BZ


def _geom(oracle, sigma=0.06, bz=BZ, n_sectors=1):
    from paper_1712_09416_b200 import gen
    return oracle.Geometry(n_sectors, gen.row_x().astype(np.float32), gen.TAN_HALF_ANGLE, sigma, sigma, bz)


def exact_helix(state, dx, kb=KB):
    """Closed form with asin (not used by the oracle): circle of curvature kappa = kb*q in (x,y), z linear in arc."""
    y, z, s, t, q = state
    kap = kb * q
    s1 = s + kap * dx
    c0, c1 = math.sqrt(1 - s * s), math.sqrt(1 - s1 * s1)
    if abs(kap) < 1e-14:
        dy = dx * s / c0
        dS = dx / c0
    else:
        dy = (c0 - c1) / kap
        dS = (math.asin(s1) - math.asin(s)) / kap
    return np.array([y + dy, z + t * dS, s1, t, q])


def mp_derivative(state, dx, k):
    """d(exact helix)/d(state_k) with 40-digit arithmetic (the closed form cancels badly in double)."""
    import mpmath as mp
    mp.mp.dps = 40

    def prop(v):
        st = [mp.mpf(float(a)) for a in state]
        st[k] = v
        y, z, s, t, q = st
        kap = mp.mpf(KB) * q
        s1 = s + kap * dx
        c0, c1 = mp.sqrt(1 - s * s), mp.sqrt(1 - s1 * s1)
        return [y + (c0 - c1) / kap, z + t * (mp.asin(s1) - mp.asin(s)) / kap, s1, t, q]

    return [mp.diff(lambda v, i=i: prop(v)[i], mp.mpf(float(state[k]))) for i in range(5)]


def random_states(rng, n):
    out = []
    while len(out) < n:
        s = rng.uniform(-0.8, 0.8); q = rng.uniform(-10, 10)
        dx = rng.choice([0.75, -0.75, 1.0, -1.0, 1.5, -1.5, 3.0, -7.5, 7.5])
        if abs(s + KB * q * dx) > 0.9:
            continue
        out.append((np.array([rng.uniform(-40, 40), rng.uniform(-250, 250), s, rng.uniform(-1.1, 1.1), q]), dx))
    return out


def test_transport_equals_exact_helix(oracle_mod):
    g = _geom(oracle_mod)
    rng = np.random.default_rng(1)
    worst = 0.0
    for st, dx in random_states(rng, 3000):
        ok, new, _ = oracle_mod.transport(g, 100.0, 100.0 + dx, st, np.eye(5))
        assert ok
        ref = exact_helix(st, dx)
        worst = max(worst, np.max(np.abs(new[:2] - ref[:2])))
        assert abs(new[2] - ref[2]) < 1e-14 and new[3] == st[3] and new[4] == st[4]
    assert worst < 1e-6, worst          # cm; series for the arc length, SURVEY.md 8(c).2


def test_transport_fails_beyond_sin_max(oracle_mod):
    g = _geom(oracle_mod)
    st = np.array([0.0, 0.0, 0.9, 0.3, -10.0])    # kappa = +0.015: sin phi grows by 0.1125 over 7.5 cm
    ok, new, cov = oracle_mod.transport(g, 100.0, 107.5, st, np.eye(5))
    assert not ok and np.array_equal(new, st) and np.array_equal(cov, np.eye(5))
    ok, _, _ = oracle_mod.transport(g, 100.0, 103.0, st, np.eye(5))
    assert ok


@pytest.mark.parametrize("precision", ["double", "float"])
def test_transport_fails_when_it_starts_beyond_sin_max(oracle_mod, precision):
    """DESIGN.md reading R9: the step fails when |sin phi| is beyond s_max at EITHER end.  Here only the START is
    beyond it (|s| = 0.96 > 0.95; an update can leave the fit there) while the step leads back inside
    (|s1| = 0.940): fit and covariance must stay untouched.  Kills the mutant of oracle/tpc_oracle.cpp `transport` that
    drops its first guard (`|s| > s_max`), which the case above (only |s1| beyond the limit) cannot see."""
    g = _geom(oracle_mod)
    cov = np.diag([0.01, 0.02, 0.003, 0.004, 0.5])
    for sign in (1.0, -1.0):
        st = np.array([1.0, -2.0, sign * 0.96, 0.3, sign * 10.0])   # kappa = -+0.015: |sin phi| falls by 0.02 over 4/3 cm
        dx = 4.0 / 3.0
        assert 0.93 < abs(st[2] + KB * st[4] * dx) < 0.945          # the far end is inside the limit
        ok, new, cn = oracle_mod.transport(g, 100.0, 100.0 + dx, st, cov, precision=precision)
        assert not ok and np.array_equal(new, st) and np.array_equal(cn, cov)
        # the same step from just inside the limit is taken (the guard is |s| > s_max, not the direction of the step)
        st[2] = sign * 0.949
        ok, new, _ = oracle_mod.transport(g, 100.0, 100.0 + dx, st, cov, precision=precision)
        assert ok and abs(new[2] - (st[2] + KB * st[4] * dx)) < 1e-6 and abs(new[2]) < 0.93


def test_jacobian_equals_central_differences_of_exact_helix(oracle_mod):
    """C' = F C F^T with C = e_k e_k^T gives column k of F in column k of C' (F_kk = 1)."""
    g = _geom(oracle_mod)
    rng = np.random.default_rng(2)
    for st, dx in random_states(rng, 60):
        F = np.zeros((5, 5))
        for k in range(5):
            E = np.zeros((5, 5)); E[k, k] = 1.0
            ok, _, Cn = oracle_mod.transport(g, 120.0, 120.0 + dx, st, E)
            assert ok
            F[:, k] = Cn[:, k]
            assert np.allclose(Cn, np.outer(Cn[:, k], Cn[:, k]), rtol=1e-12, atol=1e-15)
        num = np.zeros((5, 5))
        for k in range(5):
            num[:, k] = [float(v) for v in mp_derivative(st, dx, k)]
        scale = np.maximum(np.abs(num), 1e-6)
        err = np.abs(F - num) / scale
        exact_entries = [(i, j) for i in range(5) for j in range(5) if (i, j) != (1, 4)]
        for (i, j) in exact_entries:
            assert err[i, j] < 2e-6 or abs(F[i, j] - num[i, j]) < 1e-8, ((i, j), F[i, j], num[i, j])
        # dz/dq uses the chord approximation: within 5 % of the true derivative
        assert abs(F[1, 4] - num[1, 4]) <= 0.05 * abs(num[1, 4]) + 1e-7, (F[1, 4], num[1, 4])


def test_covariance_transport_is_F_C_Ft(oracle_mod):
    g = _geom(oracle_mod)
    rng = np.random.default_rng(3)
    for st, dx in random_states(rng, 50):
        A = rng.normal(size=(5, 5)); C0 = A @ A.T
        F = np.zeros((5, 5))
        for k in range(5):
            E = np.zeros((5, 5)); E[k, k] = 1.0
            F[:, k] = oracle_mod.transport(g, 90.0, 90.0 + dx, st, E)[2][:, k]
        _, _, C1 = oracle_mod.transport(g, 90.0, 90.0 + dx, st, C0)
        assert np.allclose(C1, F @ C0 @ F.T, rtol=1e-12, atol=1e-12)
        assert np.array_equal(C1, C1.T)


def test_update_equals_textbook_joint_kalman_update(oracle_mod):
    g = _geom(oracle_mod, sigma=0.08)
    rng = np.random.default_rng(4)
    H = np.zeros((2, 5)); H[0, 0] = 1; H[1, 1] = 1
    V = np.eye(2) * 0.08 ** 2
    V = np.diag([np.float32(0.08).astype(np.float64) ** 2] * 2)
    for _ in range(100):
        A = rng.normal(size=(5, 5)) * np.array([0.1, 0.1, 0.01, 0.01, 1.0])[:, None]
        C0 = A @ A.T + np.diag([1e-4, 1e-4, 1e-6, 1e-6, 1e-3])
        x0 = rng.normal(size=5); m = x0[:2] + rng.normal(size=2) * 0.1
        x1, C1, chi2 = oracle_mod.update(g, m[0], m[1], x0, C0, 1.5)
        S = H @ C0 @ H.T + V
        Kg = C0 @ H.T @ np.linalg.inv(S)
        r = m - H @ x0
        assert np.allclose(x1, x0 + Kg @ r, rtol=1e-9, atol=1e-12)
        assert np.allclose(C1, (np.eye(5) - Kg @ H) @ C0, rtol=1e-8, atol=1e-13)
        assert abs(chi2 - (1.5 + r @ np.linalg.inv(S) @ r)) < 1e-9 * max(1, chi2)
        assert np.array_equal(C1, C1.T)


# ---------- whole fits on generated single tracks ----------

def truth_state(trk, x_ref, alpha=math.radians(10.0), bz=BZ):
    """Local (y, z, sin phi, tg lambda, q/pT) of a generated track where it first crosses x_loc = x_ref."""
    pt, charge, eta, phi, vx, vy, vz = trk[:7]
    R = pt / (K * abs(bz)); h = -charge * (1 if bz >= 0 else -1)
    cx = vx - h * R * math.sin(phi); cy = vy + h * R * math.cos(phi)
    lcx = cx * math.cos(alpha) + cy * math.sin(alpha); lcy = -cx * math.sin(alpha) + cy * math.cos(alpha)
    psi0 = math.atan2(vy - cy, vx - cx)
    best = None
    for sgn in (-1.0, 1.0):
        d = R * R - (x_ref - lcx) ** 2
        if d <= 0:
            continue
        y = lcy + sgn * math.sqrt(d)
        psi = math.atan2(y - lcy, x_ref - lcx) + alpha
        th = (h * (psi - psi0)) % (2 * math.pi)
        if best is None or th < best[0]:
            best = (th, y)
    th, y = best
    t = math.sinh(eta)
    return np.array([y, vz + t * R * th, h * (x_ref - lcx) / R, t, charge / pt])


def _single_track_events(gen, n_events, sigma, pt_a, pt_b, ineff=0.0, bz=BZ, n_trk=1):
    out = []
    for e in range(n_events):
        r = gen.Recipe("single", n_sectors=1, n_primaries=n_trk, pt_mode=0, pt_a=pt_a, pt_b=pt_b, sigma=sigma,
                       inefficiency=ineff, noise_frac=0.0, bz=bz, config_id=50)
        out.append(gen.generate(r, event=e))
    return out


def test_noise_free_helix_is_recovered(oracle_mod, gen_mod):
    used = 0
    for ev in _single_track_events(gen_mod, 16, sigma=0.0, pt_a=0.25, pt_b=3.0):
        if ev.n_clusters < 60:          # a soft track aimed at the sector centre can curl out of the wedge
            continue
        used += 1
        g = oracle_mod.Geometry(1, gen_mod.row_x().astype(np.float32), gen_mod.TAN_HALF_ANGLE, 0.06, 0.06, BZ)
        res = oracle_mod.track_event(g, ev.sector_offset, ev.y, ev.z, ev.row, precision="double")
        assert res.n_tracks == 1
        assert res.trk_n_hits[0] == ev.n_clusters           # every hit of the track, nothing else
        tr = truth_state(ev.tracks[0], res.trk_x[0])
        fit = np.array([res.trk_y[0], res.trk_z[0], res.trk_sinphi[0], res.trk_tgl[0], res.trk_qpt[0]])
        # float32 storage of the hits (4e-6 cm) is the only noise
        assert np.all(np.abs(fit - tr) < np.array([2e-5, 4e-5, 2e-6, 2e-6, 2e-4])), (fit, tr)
        assert res.trk_chi2[0] < 1e-4
    assert used >= 8


def test_straight_line_limit_equals_weighted_least_squares(oracle_mod, gen_mod):
    """Bz -> 0: the model is linear in (y0, tan phi) and (z0, tg lambda / cos phi); the KF (a recursive least
    squares) must land on the textbook least-squares line through the hits."""
    bz = 1e-7
    for ev in _single_track_events(gen_mod, 10, sigma=0.06, pt_a=1.0, pt_b=2.0, bz=bz):
        g = oracle_mod.Geometry(1, gen_mod.row_x().astype(np.float32), gen_mod.TAN_HALF_ANGLE, 0.06, 0.06, bz)
        res = oracle_mod.track_event(g, ev.sector_offset, ev.y, ev.z, ev.row, precision="double")
        assert res.n_tracks == 1 and res.trk_n_hits[0] == ev.n_clusters
        x = ev.x.astype(np.float64); xr = res.trk_x[0]
        A = np.stack([np.ones_like(x), x - xr], axis=1)
        (y0, ty), *_ = np.linalg.lstsq(A, ev.y.astype(np.float64), rcond=None)
        (z0, tz), *_ = np.linalg.lstsq(A, ev.z.astype(np.float64), rcond=None)
        s_ls = ty / math.sqrt(1 + ty * ty)
        t_ls = tz * math.sqrt(1 - s_ls * s_ls)          # dz/dS = dz/dx * cos phi
        # statistical errors are ~1e-2 cm and ~1e-4; agreement must be far inside them
        assert abs(res.trk_y[0] - y0) < 2e-4 and abs(res.trk_z[0] - z0) < 2e-4
        assert abs(res.trk_sinphi[0] - s_ls) < 5e-6 and abs(res.trk_tgl[0] - t_ls) < 1e-5   # < 10 % of the errors
        ry = ev.y - (y0 + ty * (x - xr)); rz = ev.z - (z0 + tz * (x - xr))
        chi2_ls = (ry @ ry + rz @ rz) / 0.06 ** 2
        assert abs(res.trk_chi2[0] - chi2_ls) < 0.02 * chi2_ls + 0.5


@pytest.mark.parametrize("precision", ["double", "float"])
def test_pulls_chi2_and_gluckstern(oracle_mod, gen_mod, precision):
    sigma = 0.06
    pulls, chi2ndf, dq, sq = [], [], [], []
    for ev in _single_track_events(gen_mod, 40, sigma=sigma, pt_a=1.0, pt_b=4.0, ineff=0.02, n_trk=10):
        g = oracle_mod.Geometry(1, gen_mod.row_x().astype(np.float32), gen_mod.TAN_HALF_ANGLE, sigma, sigma, BZ)
        res = oracle_mod.track_event(g, ev.sector_offset, ev.y, ev.z, ev.row, precision=precision)
        for i in range(res.n_tracks):
            hits = res.hit_idx[res.trk_first_hit[i]:res.trk_first_hit[i] + res.trk_n_hits[i]]
            lab = ev.label[hits]
            if res.trk_n_hits[i] < 150 or np.any(lab != lab[0]):
                continue
            tr = truth_state(ev.tracks[lab[0]], res.trk_x[i])
            fit = np.array([res.trk_y[i], res.trk_z[i], res.trk_sinphi[i], res.trk_tgl[i], res.trk_qpt[i]])
            cov = res.tl_cov[res.trk_seed[i]]
            pulls.append((fit - tr) / np.sqrt(cov))
            chi2ndf.append(res.trk_chi2[i] / res.trk_ndf[i])
            dq.append(fit[4] - tr[4]); sq.append(math.sqrt(cov[4]))
    pulls = np.array(pulls)
    assert pulls.shape[0] > 200
    assert np.all(np.abs(pulls.mean(axis=0)) < 0.15), pulls.mean(axis=0)
    rms = pulls.std(axis=0)
    assert np.all((rms > 0.85) & (rms < 1.15)), rms
    assert 0.9 < np.mean(chi2ndf) < 1.1, np.mean(chi2ndf)
    # Gluckstern: sigma_kappa = sigma / L^2 * sqrt(720 / (N + 4)), sigma(q/pT) = sigma_kappa / (K Bz)
    N, L = 155, 245.85 - 85.225
    gl = sigma / L ** 2 * math.sqrt(720.0 / (N + 4)) / (K * BZ)
    assert 0.75 * gl < np.std(dq) < 1.35 * gl, (np.std(dq), gl)
    assert 0.75 * gl < np.mean(sq) < 1.35 * gl, (np.mean(sq), gl)
