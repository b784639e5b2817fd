"""Pins for the oracle's floating-point stage (transport, Jacobian, update, follower) and stage 5.
Each pin is something the mathematics fixes independently of the oracle's own formulas (SURVEY 8c pin table)."""
import numpy as np
import pytest

from gen.events import make_event, truth_params_at
from gen.rng import Rng
from gen.truth import match_tracks

CQ = -0.00299792458 * 0.5


def _states(n, seed=5):
    r = Rng(seed)
    y = r.uniform(1, n) * 80 - 40
    z = r.uniform(2, n) * 500 - 250
    s = r.uniform(3, n) * 1.6 - 0.8
    t = r.uniform(4, n) * 2 - 1
    q = (r.uniform(5, n) * 2 - 1) * 10
    return np.stack([y, z, s, t, q], axis=1)


def test_transport_keeps_circle_centre_and_pitch(orc):
    """Geometry pin: a circle with tangent (cos phi, sin phi) and signed curvature k has its centre at
    (x, y) + (-sin phi, cos phi)/k; transport along the circle must not move the centre, and z advances by
    tan(lambda) times the arc length (phi1 - phi0)/k."""
    for st in _states(200):
        for dx in (1.0596, -1.0596, 5.3, -0.3):
            k = CQ * st[4]
            ok, s1, _ = orc.transport(st, None, dx, CQ, sinphi_max=0.999)
            if not ok:
                continue
            c0, c1 = np.sqrt(1 - st[2] ** 2), np.sqrt(1 - s1[2] ** 2)
            cen0 = np.array([0.0 - st[2] / k, st[0] + c0 / k])
            cen1 = np.array([dx - s1[2] / k, s1[0] + c1 / k])
            assert np.allclose(cen0, cen1, rtol=0, atol=1e-9 * max(1.0, abs(1 / k)))
            arc = (np.arcsin(s1[2]) - np.arcsin(st[2])) / k
            assert abs((s1[1] - st[1]) - st[3] * arc) < 1e-9 * max(1.0, abs(arc))
            assert s1[3] == st[3] and s1[4] == st[4]
            assert abs(s1[2] - (st[2] + k * dx)) < 1e-15


def test_transport_closed_form_dy(orc):
    st = np.array([1.0, 2.0, 0.3, 0.5, 2.0])
    k = CQ * st[4]
    ok, s1, _ = orc.transport(st, None, 10.0, CQ)
    assert ok
    assert abs((s1[0] - st[0]) - (np.sqrt(1 - 0.3 ** 2) - np.sqrt(1 - s1[2] ** 2)) / k) < 1e-10


def test_transport_straight_line_limit(orc):
    """q/pT = 0: straight line y += dx tan(phi), z += tan(lambda) dx / cos(phi)."""
    st = np.array([1.0, -2.0, 0.6, 0.7, 0.0])
    ok, s1, _ = orc.transport(st, None, 3.0, CQ)
    assert ok and abs(s1[0] - (1.0 + 3.0 * 0.6 / 0.8)) < 1e-14 and abs(s1[1] - (-2.0 + 0.7 * 3.0 / 0.8)) < 1e-14


def test_transport_reversible_and_fails_at_sinphi_max(orc):
    for st in _states(100, seed=6):
        ok, s1, _ = orc.transport(st, None, 2.5, CQ, 0.999)
        if not ok:
            continue
        ok2, s2, _ = orc.transport(s1, None, -2.5, CQ, 0.999)
        assert ok2 and np.allclose(s2, st, rtol=0, atol=1e-12)
    st = np.array([0.0, 0.0, 0.9499, 0.0, -10.0])        # k > 0: sin phi grows
    assert orc.transport(st, None, 1.0, CQ)[0] is False  # s1 = 0.9499 + 0.015 >= 0.95
    assert orc.transport(st, None, -1.0, CQ)[0] is True
    st[2] = 0.95
    assert orc.transport(st, None, -1.0, CQ)[0] is False  # |sin phi| >= 0.95 before the step


def test_jacobian_matches_central_differences(orc):
    for st in _states(60, seed=7):
        for dx in (1.0596, -3.0):
            if abs(st[2] + CQ * st[4] * dx) > 0.9 or abs(st[2]) > 0.9:
                continue
            F = orc.jacobian(st, dx, CQ)
            Fd = np.zeros((5, 5))
            for j in range(5):
                h = 1e-6 * max(1.0, abs(st[j]))
                a, b = st.copy(), st.copy()
                a[j] += h
                b[j] -= h
                Fd[:, j] = (orc.transport(a, None, dx, CQ, 0.9999)[1] - orc.transport(b, None, dx, CQ, 0.9999)[1]) / (2 * h)
            assert np.allclose(F, Fd, rtol=2e-7, atol=2e-7), (st, dx, F - Fd)


def test_dz_dq_matches_long_double_closed_form(orc):
    """d(dS)/dk = (dx/c1 - dS)/k with dS = (asin s1 - asin s)/k, evaluated in 80-bit long double where the
    subtraction is still well conditioned; pins the series / stable form used for small k."""
    L = np.longdouble
    for (s, q, dx) in [(0.3, 1.0, 1.06), (-0.7, 8.0, 1.06), (0.0, 0.05, 1.06), (0.5, -0.5, -4.0), (0.2, 20.0, 5.0)]:
        st = np.array([0.0, 0.0, s, 0.8, q])
        F = orc.jacobian(st, dx, CQ)
        k = L(CQ) * L(q)
        s1 = L(s) + k * L(dx)
        dS = (np.arcsin(s1) - np.arcsin(L(s))) / k
        dSdk = (L(dx) / np.sqrt(1 - s1 * s1) - dS) / k
        ref = float(L(0.8) * L(CQ) * dSdk)
        assert abs(F[1, 4] - ref) <= 1e-9 * abs(ref) + 1e-15, (s, q, dx, F[1, 4], ref)
    # k -> 0 limit: dS'(k) -> dx^2 s / (2 c^3)
    st = np.array([0.0, 0.0, 0.4, 1.0, 0.0])
    F = orc.jacobian(st, 2.0, CQ)
    assert abs(F[1, 4] - CQ * 4.0 * 0.4 / (2 * (1 - 0.16) ** 1.5)) < 1e-15


def test_covariance_transport_is_F_C_Ft(orc):
    st = np.array([3.0, -20.0, 0.4, -0.6, 3.0])
    A = np.arange(25, dtype=float).reshape(5, 5) / 10 + np.eye(5)
    C = A @ A.T
    F = orc.jacobian(st, 1.0596, CQ)
    ok, _, C1 = orc.transport(st, C, 1.0596, CQ)
    assert ok and np.allclose(C1, F @ C @ F.T, rtol=1e-13, atol=0)


def test_update_equals_information_form(orc):
    """Textbook identity: posterior = (C^-1 + H^T V^-1 H)^-1, mean = C'(C^-1 p + H^T V^-1 m)."""
    r = Rng(9)
    for i in range(20):
        A = r.uniform(10 + i, 25).reshape(5, 5) - 0.5
        C = A @ A.T + 0.1 * np.eye(5)
        p = r.uniform(40 + i, 5) * 2 - 1
        m = r.uniform(70 + i, 2) * 2 - 1
        V = np.diag([0.01, 0.0225])
        H = np.zeros((2, 5))
        H[0, 0] = H[1, 1] = 1
        Ci = np.linalg.inv(C)
        Cp = np.linalg.inv(Ci + H.T @ np.linalg.inv(V) @ H)
        pp = Cp @ (Ci @ p + H.T @ np.linalg.inv(V) @ m)
        st, cov, chi2 = orc.update(p, C, m[0], m[1], 0.01, 0.0225)
        assert np.allclose(st, pp, rtol=1e-9, atol=1e-11) and np.allclose(cov, Cp, rtol=1e-8, atol=1e-11)
        res = m - p[:2]
        assert abs(chi2 - res @ np.linalg.inv(C[:2, :2] + V) @ res) < 1e-9 * max(1, chi2)
        assert np.array_equal(cov, cov.T)


def test_straight_line_filter_equals_least_squares(orc):
    """Bz -> 0 with a diffuse prior and tiny noise: the filter over a row sequence equals the straight-line
    least-squares fit (numpy lstsq) of y(x) and z(x)."""
    r = Rng(11)
    xs = 85 + np.arange(40) * (160.0 / 151)
    a, b, c, d = 3.0, 0.2, -10.0, 0.5            # y = a + b (x-x0), z = c + d (x-x0)
    ym = a + b * (xs - xs[0]) + 1e-4 * r.normal(1, 40)
    zm = c + d * (xs - xs[0]) + 1e-4 * r.normal(2, 40)
    st = np.array([ym[0], zm[0], b / np.hypot(1, b), d / np.hypot(1, b), 0.0])
    C = np.diag([1e2, 1e2, 1.0, 1.0, 1.0])
    st, C, _ = orc.update(st, C, ym[0], zm[0], 1e-8, 1e-8)
    for i in range(1, 40):
        ok, st, C = orc.transport(st, C, xs[i] - xs[i - 1], 0.0)
        assert ok
        st, C, _ = orc.update(st, C, ym[i], zm[i], 1e-8, 1e-8)
    A = np.stack([np.ones(40), xs - xs[-1]], axis=1)
    (y_end, slope_y), *_ = np.linalg.lstsq(A, ym, rcond=None)
    (z_end, slope_z), *_ = np.linalg.lstsq(A, zm, rcond=None)
    cosphi = np.sqrt(1 - st[2] ** 2)
    assert abs(st[0] - y_end) < 1e-7 and abs(st[1] - z_end) < 1e-7
    assert abs(st[2] / cosphi - slope_y) < 1e-7 and abs(st[3] / cosphi - slope_z) < 1e-7
    assert st[4] == 0.0


def _truth_errors(ev, o):
    errs = []
    for i, t in enumerate(o["trk_seed"]):
        h0 = o["hit_ids"][o["trk_hit_offset"][i]]
        trk = ev.label[h0] // 64
        par = o["par"][t]
        tp = truth_params_at(ev, trk, 0, par[0])
        errs.append(np.abs(par[1:] - tp) / np.maximum(np.abs(tp), 1.0))
    return np.array(errs)


def test_exact_helices_reconstructed_to_1e4(orc):
    """north_star pin: noise-free, zero-smearing helices -> 100 % efficiency, fitted parameters = truth to 1e-4
    (exact doubles fed to the follower, bypassing quantisation)."""
    ev = make_event(0, sigma_scale=0.0)
    o = orc.track(ev, exact_coords=True)
    m = match_tracks(ev, np.zeros(len(o["trk_seed"]), dtype=int), o["trk_hit_offset"], o["trk_n_owned"], o["hit_ids"])
    assert m["n_out"] == 100 and m["efficiency"] == 1.0 and m["n_fake"] == 0 and m["n_clone"] == 0
    assert _truth_errors(ev, o).max() < 1e-4
    assert _truth_errors(ev, o).max() < 2e-5          # what the method actually reaches (9e-6)


def test_quantised_helices_through_int32(orc):
    """Same through the int32 interface: 1e-4 for sin phi, tan lambda, q/pT; one quantum (1/640 cm) floor for
    y and z (P37: +-1/2-quantum input rounding alone moves y by ~1e-4 cm)."""
    ev = make_event(0, sigma_scale=0.0)
    o = orc.track(ev)
    e = _truth_errors(ev, o)
    assert len(o["trk_seed"]) == 100
    assert e[:, 2:].max() < 1e-4 and e[:, :2].max() < 1.0 / 640


def test_nominal_config0_efficiency(orc):
    ev = make_event(0)
    o = orc.track(ev)
    m = match_tracks(ev, np.zeros(len(o["trk_seed"]), dtype=int), o["trk_hit_offset"], o["trk_n_owned"], o["hit_ids"])
    assert m["efficiency"] == 1.0 and m["n_fake"] == 0


def test_search_modes_agree(orc):
    """Full-row scan (the definition, P17) == z-sorted pruning."""
    ev = make_event(4, n_tracks=250)
    a = orc.track(ev, search_mode=0)
    b = orc.track(ev, search_mode=1)
    assert np.array_equal(a["hits"], b["hits"]) and np.array_equal(a["par"], b["par"])


def test_mirror_symmetry(orc):
    """y -> -y with q -> -q: mirrored tracks, same hit lists (pins the curvature-sign convention P4)."""
    ev = make_event(0)
    a = orc.track(ev)
    ev2 = make_event(0)
    ev2.y = (-ev2.y).astype(np.int32)
    b = orc.track(ev2)
    assert np.array_equal(a["hits"], b["hits"]) and np.array_equal(a["hit_ids"], b["hit_ids"])
    sign = np.array([1, -1, 1, -1, 1, -1.0])
    assert np.allclose(a["par"] * sign, b["par"], rtol=1e-9, atol=1e-11)


def test_z_translation_shifts_only_z(orc):
    ev = make_event(0)
    a = orc.track(ev)
    ev2 = make_event(0)
    ev2.z = ev2.z + np.int32(640 * 1000)
    b = orc.track(ev2)
    assert np.array_equal(a["hits"], b["hits"])
    shift = np.zeros(6)
    shift[2] = 1000.0
    assert np.allclose(a["par"] + shift, b["par"], rtol=0, atol=1e-8)


def test_selection_invariants(orc):
    ev = make_event(4, n_tracks=400)
    o = orc.track(ev)
    sec, row = ev.sector_row()
    # each cluster appears in at most one output list and is owned by that track's seed
    ids = o["hit_ids"]
    assert len(np.unique(ids)) == len(ids)
    for t in range(len(o["trk_seed"])):
        h = ids[o["trk_hit_offset"][t]: o["trk_hit_offset"][t] + o["trk_n_owned"][t]]
        assert np.all(o["owner"][h] == o["trk_seed"][t])
        assert np.all(np.diff(row[h]) > 0)                         # ascending row, <= 1 hit per row
        assert len(h) >= 10
        assert len(set(sec[h])) == 1
    assert np.all(np.diff(o["seed_start"][o["trk_seed"]]) > 0)     # output order = ascending seed start id
    # ownership rule on a hand-made contest: longer tracklet wins, ties -> smaller start id
    hits = np.full((3, 12), -1, dtype=np.int32)
    hits[0, :10] = np.arange(10)               # tracklet 0: clusters 0..9
    hits[1, :11] = np.arange(5, 16)            # tracklet 1: clusters 5..15 (11 hits) -> wins 5..9
    hits[2, :11] = np.arange(5, 16)            # tracklet 2: same length as 1, larger start id -> loses all
    n_hits = np.array([10, 11, 11], dtype=np.int32)
    p = orc.default_params()
    p.n_min_owned = 1
    owner, trk_seed, trk_n, trk_off, hit_ids = orc.select(16, 12, np.array([0, 5, 6], dtype=np.int32), n_hits, hits, p)
    assert owner.tolist() == [0] * 5 + [1] * 11
    assert trk_seed.tolist() == [0, 1] and trk_n.tolist() == [5, 11]
    assert hit_ids.tolist() == list(range(5)) + list(range(5, 16))


# ---- NEXT-1: refit of output tracks over their owned hits (orc_refit, reading P41) ----

def _refit_truth_errors(ev, o):
    errs = []
    for i in range(len(o["trk_seed"])):
        h0 = o["hit_ids"][o["trk_hit_offset"][i]]
        par = o["refit_par"][i]
        tp = truth_params_at(ev, ev.label[h0] // 64, 0, par[0])
        errs.append(np.abs(par[1:] - tp) / np.maximum(np.abs(tp), 1.0))
    return np.array(errs)


def test_refit_exact_helices_to_1e4(orc):
    """Pin by the problem: on noise-free exact helices the refit over the owned hits gives the generator's truth
    parameters at the lowest owned hit to 1e-4 (a wrong gap dx, a dropped update or a wrong pass order fails)."""
    ev = make_event(0, sigma_scale=0.0)
    o = orc.track(ev, exact_coords=True)
    assert len(o["refit_par"]) == 100
    assert np.array_equal(o["refit_used"], o["trk_n_owned"])          # every owned hit is used on the way down
    assert _refit_truth_errors(ev, o).max() < 2e-5


def test_refit_with_row_gaps_still_reaches_truth(orc):
    """Owned hit lists with gaps (every third hit removed): transports over several rows at once; the truth pin
    still holds, so the gap dx is taken from the row positions of the hits, not from a fixed pitch."""
    ev = make_event(0, sigma_scale=0.0)
    o = orc.track(ev, exact_coords=True)
    keep, off, cnt = [], [], []
    for i in range(len(o["trk_seed"])):
        h = o["hit_ids"][o["trk_hit_offset"][i]: o["trk_hit_offset"][i] + o["trk_n_owned"][i]]
        h = np.delete(h, np.arange(2, len(h), 3))
        off.append(sum(cnt))
        cnt.append(len(h))
        keep.append(h)
    hit_ids = np.concatenate(keep).astype(np.int32)
    par, cov, chi2, used = orc.refit(ev.y_exact, ev.z_exact, ev.row_offsets, ev.n_sectors, ev.n_rows, ev.row_x,
                                     ev.cfg.bz, np.array(off, np.int32), np.array(cnt, np.int32), hit_ids)
    o2 = dict(o, refit_par=par, hit_ids=hit_ids, trk_hit_offset=np.array(off))
    assert np.array_equal(used, np.array(cnt))
    assert _refit_truth_errors(ev, o2).max() < 2e-5


def test_refit_equals_tracklet_fit_on_full_length_tracks(orc):
    """Pin against the (independently pinned) follower: for a tracklet that has a hit in every row from 0 to the last
    row and owns all of them, the follower's downward pass (after the covariance reset) runs over exactly the hits
    of the refit's downward pass.  The upward passes differ only in where they start (the seed starts in row 1: rows
    0 and n-1 have no links of their own, P5), which moves the linearisation point of the downward pass by ~1e-9,
    so the two fits agree to 1e-8 -- and not to more if the refit dropped or reordered a hit."""
    ev = make_event(0, sigma_scale=0.0)
    o = orc.track(ev, exact_coords=True)
    n = 0
    for i, t in enumerate(o["trk_seed"]):
        if o["trk_n_owned"][i] == ev.n_rows and (o["hits"][t] >= 0).all():
            assert np.allclose(o["refit_par"][i], o["par"][t], rtol=0, atol=1e-8)
            assert np.allclose(o["refit_cov"][i], o["cov"][t], rtol=1e-6, atol=1e-15)
            assert abs(o["refit_chi2"][i] - o["chi2"][t]) < 1e-8
            n += 1
    assert n >= 20


def test_refit_nominal_config_improves_nothing_it_should_not(orc):
    """Sanity on smeared data: chi2 per degree of freedom of the refit is ~1 (errors sigma_y, sigma_z are the true
    smearing in configs[0]) -- a transposed gain or a wrong V would move it far away."""
    ev = make_event(0)
    o = orc.track(ev)
    ndf = 2 * o["refit_used"] - 5
    ok = ndf > 20
    r = o["refit_chi2"][ok] / ndf[ok]
    assert 0.8 < np.median(r) < 1.2
