"""Pins for the oracle's NEXT-1 merging step (readings P42..P46): frame rotation between sectors, the
match chi2 and the mutual-best link rule.  Expected values come from plane geometry worked out here, from the
generator's global helices (gen/, independent of the tracker's parametrisation) and from hand-made records."""
import numpy as np
import pytest

from gen.events import make_event, truth_params_at
from gen.rng import Rng

CQ = -0.00299792458 * 0.5
A20 = np.deg2rad(20.0)


def _spd(seed, scale):
    r = Rng(seed)
    a = r.uniform(1, 25).reshape(5, 5) - 0.5
    c = a @ a.T + 0.5 * np.eye(5)
    d = np.asarray(scale)
    return c * d[:, None] * d[None, :]


def _pack(c):
    return np.array([c[i, j] for i in range(5) for j in range(i + 1)])


def test_rotation_is_plane_geometry(orc):
    """The same point and direction seen from a frame turned by alpha: x' = x cos a + y sin a, y' = -x sin a + y cos a,
    phi' = phi - a; z, tan lambda and q/pT do not change."""
    for (x, y, phi, alpha) in [(100.0, 10.0, 0.3, A20), (150.0, -30.0, -0.2, -A20), (90.0, 5.0, 0.0, 0.1)]:
        st = np.array([y, -7.0, np.sin(phi), 0.6, 1.5])
        ok, x1, s1, _ = orc.rotate(x, st, None, alpha, CQ)
        assert ok
        assert abs(x1 - (x * np.cos(alpha) + y * np.sin(alpha))) < 1e-12
        assert abs(s1[0] - (-x * np.sin(alpha) + y * np.cos(alpha))) < 1e-12
        assert abs(s1[2] - np.sin(phi - alpha)) < 1e-14
        assert s1[1] == st[1] and s1[3] == st[3] and s1[4] == st[4]


def test_rotation_there_and_back_is_identity(orc):
    st = np.array([12.0, -40.0, 0.35, -0.7, 2.0])
    C = _spd(3, [0.1, 0.2, 0.01, 0.01, 0.05])
    ok, x1, s1, C1 = orc.rotate(120.0, st, C, A20, CQ)
    ok2, x2, s2, C2 = orc.rotate(x1, s1, C1, -A20, CQ)
    assert ok and ok2 and abs(x2 - 120.0) < 1e-11
    assert np.allclose(s2, st, rtol=0, atol=1e-12) and np.allclose(C2, C, rtol=1e-11, atol=1e-16)


def test_rotation_fails_when_the_track_does_not_move_along_the_new_x(orc):
    st = np.array([0.0, 0.0, 0.94, 0.0, 0.0])           # phi = 70 deg
    assert orc.rotate(100.0, st, None, -A20, CQ)[0] is False     # phi' = 90 deg: |sin phi'| >= 0.95
    assert orc.rotate(100.0, st, None, A20, CQ)[0] is True       # phi' = 50 deg
    st[2] = -0.94
    assert orc.rotate(100.0, st, None, A20, CQ)[0] is False


def test_rotate_and_transport_follow_the_generator_helix_into_the_next_sector(orc):
    """Truth parameters of a generated helix in sector s, rotated by +20 degrees and transported, must be the
    generator's truth parameters in sector s + 1 (global-helix expressions of gen/, Appendix D)."""
    ev = make_event(1, 5, n_tracks=300, noise=0.0)
    n = 0
    for trk in range(300):
        for s in range(18):
            pa = truth_params_at(ev, trk, s, 140.0)
            pb = truth_params_at(ev, trk, s + 1, 170.0)
            if not (np.all(np.isfinite(pa)) and np.all(np.isfinite(pb))):
                continue
            if abs(pa[2]) > 0.6 or abs(pb[2]) > 0.6 or abs(pa[0]) > 60 or abs(pb[0]) > 60:
                continue
            if ev.truth["side"][trk] != 0:
                continue
            ok, x1, s1, _ = orc.rotate(140.0, pa, None, A20, CQ)
            ok2, s2, _ = orc.transport(s1, None, 170.0 - x1, CQ)
            if not (ok and ok2):
                continue
            # same helix leg (the generator picks the outgoing branch in both frames)
            if abs(s2[1] - pb[1]) > 1.0:
                continue
            assert np.allclose(s2, pb, rtol=0, atol=2e-9 * max(1.0, abs(1.0 / (CQ * pa[4])))), (trk, s, s2, pb)
            n += 1
    assert n >= 50


def test_rotation_jacobian_by_finite_differences(orc):
    """Covariance through rotate + transport to a fixed plane equals J C J^T with J the central-difference Jacobian of
    that composite map (the transport Jacobian is pinned on its own in test_oracle_kalman.py)."""
    st = np.array([8.0, -25.0, 0.30, 0.8, 3.0])
    x0, xt = 130.0, 160.0

    def g(s):
        ok, x1, s1, _ = orc.rotate(x0, s, None, A20, CQ, 0.999)
        ok2, s2, _ = orc.transport(s1, None, xt - x1, CQ, 0.999)
        assert ok and ok2
        return s2

    J = np.zeros((5, 5))
    for j in range(5):
        h = 1e-6 * max(1.0, abs(st[j]))
        a, b = st.copy(), st.copy()
        a[j] += h
        b[j] -= h
        J[:, j] = (g(a) - g(b)) / (2 * h)
    C = _spd(7, [0.05, 0.08, 0.004, 0.006, 0.03])
    ok, x1, s1, C1 = orc.rotate(x0, st, C, A20, CQ)
    ok2, s2, C2 = orc.transport(s1, C1, xt - x1, CQ)
    assert ok and ok2
    ref = J @ C @ J.T
    assert np.allclose(C2, ref, rtol=2e-6, atol=1e-12), np.abs(C2 - ref).max()


# ------------------------------------------------------------------------------------------ match chi2 and link rule
def _line_record(sector_frame_angle, x_ref, p0, d, z0, tz):
    """Record (x_ref, y, z, sin phi, tan lambda, 0) of the straight line through global point p0 with global direction
    angle d (radians), seen in a frame whose x axis points at `sector_frame_angle`, at local x = x_ref."""
    ca, sa = np.cos(sector_frame_angle), np.sin(sector_frame_angle)
    px, py = p0[0] * ca + p0[1] * sa, -p0[0] * sa + p0[1] * ca
    phi = d - sector_frame_angle
    t = (x_ref - px) / np.cos(phi)                  # path length in the xy plane from p0
    y = py + t * np.sin(phi)
    return np.array([x_ref, y, z0 + tz * t, np.sin(phi), tz, 0.0])


def _cov_small():
    return _pack(np.diag([0.01, 0.02, 1e-4, 1e-4, 1e-2]))


def test_match_chi2_is_zero_for_the_same_line_seen_from_two_sectors(orc):
    p0, d = (60.0, 30.0), np.deg2rad(35.0)
    a = _line_record(np.deg2rad(30.0), 120.0, p0, d, 5.0, 0.4)      # sector azimuth 30 deg
    b = _line_record(np.deg2rad(50.0), 170.0, p0, d, 5.0, 0.4)      # next sector, 50 deg
    c = orc.match_chi2(a, _cov_small(), b, _cov_small(), A20, CQ)
    assert 0.0 <= c < 1e-18
    # a known offset: y of b moved by 0.3 cm -> chi2 = 0.09 / (Cyy_a' + Cyy_b) with everything else uncorrelated?
    # not diagonal after transport, so compare with the explicit 5x5 solve done here
    b2 = b.copy()
    b2[1] += 0.3
    ok, x1, s1, C1 = orc.rotate(a[0], a[1:], np.diag([0.01, 0.02, 1e-4, 1e-4, 1e-2]), A20, CQ)
    ok2, s2, C2 = orc.transport(s1, C1, b[0] - x1, CQ)
    S = C2 + np.diag([0.01, 0.02, 1e-4, 1e-4, 1e-2])
    D = b2[1:] - s2
    assert abs(orc.match_chi2(a, _cov_small(), b2, _cov_small(), A20, CQ) - D @ np.linalg.solve(S, D)) < 1e-9


def _merge(orc, recs, **kw):
    par = np.array([r[0] for r in recs])
    cov = np.array([_cov_small() for _ in recs])
    sector = np.array([r[1] for r in recs], np.int32)
    first = np.array([r[2] for r in recs], np.int32)
    last = np.array([r[3] for r in recs], np.int32)
    return orc.merge(par, cov, sector, first, last, 0.5, **kw)


def test_link_needs_a_row_gap_between_1_and_gap_max(orc):
    p0, d = (60.0, 30.0), np.deg2rad(35.0)
    a = _line_record(np.deg2rad(30.0), 100.0, p0, d, 5.0, 0.4)
    b = _line_record(np.deg2rad(30.0), 150.0, p0, d, 5.0, 0.4)      # same sector: a later segment of the line
    for gap, linked in ((0, False), (1, True), (25, True), (26, False), (-3, False)):
        succ, pred, chi2, nl = _merge(orc, [(a, 1, 10, 60), (b, 1, 60 + gap, 120)])
        assert (nl == 1) == linked, gap
        if linked:
            assert succ.tolist() == [1, -1] and pred.tolist() == [-1, 0] and chi2[0] < 1e-18 and chi2[1] == -1


def test_sector_relations(orc):
    """Same sector, azimuthal neighbours on one side (with wrap-around 17 -> 0), and the sector facing across the
    central membrane are candidates; nothing else is."""
    p0, d = (60.0, 30.0), np.deg2rad(35.0)

    def rec(az_deg, x):
        return _line_record(np.deg2rad(az_deg), x, p0, d, 5.0, 0.4)

    az = lambda s: (s % 18 + 0.5) * 20.0      # noqa: E731  (P2)
    cases = [(1, 2, True), (2, 1, True), (1, 3, False), (1, 1, True), (19, 20, True), (1, 20, False), (1, 19, True),
             (17, 0, True), (0, 17, True), (35, 18, True), (0, 35, False),
             (37, 38, True), (37, 55, True), (19, 37, False), (1, 37, False)]   # second event of a batch: sectors 36..71
    for sa, sb, linked in cases:
        a, b = rec(az(sa), 100.0), rec(az(sb), 150.0)
        if abs(a[3]) > 0.9 or abs(b[3]) > 0.9:
            continue
        succ, pred, chi2, nl = _merge(orc, [(a, sa, 10, 60), (b, sb, 61, 120)])
        assert (nl == 1) == linked, (sa, sb)
    # wrap-around needs a line near azimuth 0: build it explicitly
    p0, d = (80.0, 0.0), np.deg2rad(2.0)
    a, b = _line_record(np.deg2rad(350.0), 100.0, p0, d, 0.0, 0.1), _line_record(np.deg2rad(10.0), 140.0, p0, d, 0.0, 0.1)
    assert _merge(orc, [(a, 17, 5, 40), (b, 0, 41, 80)])[3] == 1
    assert _merge(orc, [(a, 35, 5, 40), (b, 18, 41, 80)])[3] == 1


def test_mutual_best_rule_and_tie_break(orc):
    """succ(a) = argmin chi2 over its candidates, pred(b) likewise; a link stands only if both agree (P45)."""
    p0, d = (60.0, 30.0), np.deg2rad(35.0)
    a = _line_record(np.deg2rad(30.0), 100.0, p0, d, 5.0, 0.4)
    b_exact = _line_record(np.deg2rad(30.0), 150.0, p0, d, 5.0, 0.4)
    b_off = b_exact.copy()
    b_off[1] += 0.2                                   # worse match for a
    a_off = a.copy()
    a_off[1] += 0.1                                   # a second inner segment, slightly off
    # a -> {b_off, b_exact}: a picks b_exact (smaller chi2) whatever the order
    for order in ((b_off, b_exact), (b_exact, b_off)):
        succ, pred, chi2, nl = _merge(orc, [(a, 1, 10, 60), (order[0], 1, 61, 120), (order[1], 1, 61, 120)])
        want = 2 if order[1] is b_exact else 1
        assert nl == 1 and succ[0] == want and pred[want] == 0
    # {a, a_off} -> b_exact: b's best predecessor is a; a_off's only candidate is b, but b prefers a: a_off stays alone
    succ, pred, chi2, nl = _merge(orc, [(a_off, 1, 10, 60), (a, 1, 10, 60), (b_exact, 1, 61, 120)])
    assert nl == 1 and succ.tolist() == [-1, 2, -1] and pred.tolist() == [-1, -1, 1]
    # exact tie (two identical continuations): the smaller index wins
    succ, pred, chi2, nl = _merge(orc, [(a, 1, 10, 60), (b_exact, 1, 61, 120), (b_exact.copy(), 1, 61, 120)])
    assert nl == 1 and succ[0] == 1
    # chi2 cut
    far = b_exact.copy()
    far[1] += 5.0
    assert _merge(orc, [(a, 1, 10, 60), (far, 1, 61, 120)])[3] == 0
    assert _merge(orc, [(a, 1, 10, 60), (far, 1, 61, 120)], chi2_max=1e9)[3] == 1


def test_exact_helices_crossing_sector_edges_are_linked_and_only_those(orc):
    """Pin by the problem: on noise-free exact helices every link joins two segments of the same generated particle,
    and every particle that leaves a sector through its edge with both segments reconstructed is joined."""
    ev = make_event(1, 11, n_tracks=1500, noise=0.0, sigma_scale=0.0)
    o = orc.track(ev)
    s, f, l = orc.track_records(ev, o)
    def majority(a, n):                      # tracks that cross another may carry a few foreign clusters
        v, c = np.unique(ev.label[o["hit_ids"][a:a + n]] // 64, return_counts=True)
        return v[c.argmax()]

    lab = np.array([majority(a, n) for a, n in zip(o["trk_hit_offset"], o["trk_n_owned"])])
    succ, pred, chi2, nl = orc.merge(o["refit_par"], o["refit_cov"], s, f, l, ev.cfg.bz)
    a = np.nonzero(succ >= 0)[0]
    assert nl == len(a) > 400
    assert np.all(lab[a] == lab[succ[a]])                                   # purity 100 %
    assert np.all(s[a] // 18 == s[succ[a]] // 18) and np.all(f[succ[a]] > l[a])
    # completeness: pairs of tracks of one particle in neighbouring sectors with a row gap of 1..25
    want = 0
    got = 0
    order = np.argsort(lab, kind="stable")
    for k in range(len(order) - 1):
        i, j = order[k], order[k + 1]
        if lab[i] != lab[j]:
            continue
        lo, hi = (i, j) if f[i] < f[j] else (j, i)
        if 1 <= f[hi] - l[lo] <= 25 and s[lo] != s[hi]:
            want += 1
            got += int(succ[lo] == hi)
    assert want > 400 and got >= 0.99 * want, (got, want)
    # chains never branch and never loop
    assert len(set(succ[a].tolist())) == len(a)


# ------------------------------------------------------------------------------------------ P47: refit over chains
def _merged(orc, ev, o, exact=False):
    s, f, l = orc.track_records(ev, o)
    succ, pred, chi2, nl = orc.merge(o["refit_par"], o["refit_cov"], s, f, l, ev.cfg.bz)
    y, z = (ev.y_exact, ev.z_exact) if exact else (ev.y / 640.0, ev.z / 640.0)
    r = orc.refit_merged(y, z, ev.row_offsets, ev.n_sectors, ev.n_rows, ev.row_x, ev.cfg.bz, o["trk_hit_offset"],
                         o["trk_n_owned"], o["hit_ids"], succ, pred)
    return s, succ, pred, r


def test_merged_refit_of_unlinked_tracks_is_the_plain_refit(orc):
    ev = make_event(1, 21, n_tracks=600)
    o = orc.track(ev)
    s, succ, pred, (par, cov, chi2, used, osec) = _merged(orc, ev, o)
    alone = (succ < 0) & (pred < 0)
    assert alone.sum() > 100
    assert np.array_equal(par[alone], o["refit_par"][alone]) and np.array_equal(cov[alone], o["refit_cov"][alone])
    assert np.array_equal(used[alone], o["refit_used"][alone]) and np.array_equal(osec[alone], s[alone])
    assert np.all(used[pred >= 0] == 0)                               # only chain heads carry a result


def test_merged_refit_reaches_generator_truth_across_sector_edges(orc):
    """Exact helices: the fit over both pieces of a particle that crosses a sector edge uses every hit of both, and
    gives the generator's truth parameters at the first hit in the first piece's frame -- so the state was rotated by
    the right angle, in the right direction, with the right reference-plane bookkeeping, on the way up AND back."""
    ev = make_event(1, 11, n_tracks=1500, noise=0.0, sigma_scale=0.0)
    o = orc.track(ev, exact_coords=True)
    s, succ, pred, (par, cov, chi2, used, osec) = _merged(orc, ev, o, exact=True)
    heads = np.nonzero((pred < 0) & (succ >= 0))[0]
    assert len(heads) > 300
    n_hits_chain = np.array([sum(o["trk_n_owned"][c] for c in _chain(succ, a)) for a in heads])
    full = used[heads] == n_hits_chain
    assert full.mean() > 0.9                                          # the rest stop at |sin phi| >= 0.95 in a turned frame
    worst, n_pure = 0.0, 0
    for a in heads[full]:
        hits = np.concatenate([o["hit_ids"][o["trk_hit_offset"][c]: o["trk_hit_offset"][c] + o["trk_n_owned"][c]]
                               for c in _chain(succ, a)])
        lab = ev.label[hits] // 64
        if not np.all(lab == lab[0]):
            continue                       # a track that crosses another may own one of its clusters
        n_pure += 1
        tp = truth_params_at(ev, lab[0], int(s[a]), par[a, 0])
        worst = max(worst, float((np.abs(par[a, 1:] - tp) / np.maximum(np.abs(tp), 1.0)).max()))
        assert osec[a] == s[a]
    assert n_pure > 0.95 * full.sum() and worst < 5e-5, (n_pure, worst)


def _chain(succ, a):
    while a >= 0:
        yield a
        a = succ[a]


def test_merged_refit_tightens_the_fit_and_keeps_chi2_per_dof_at_one(orc):
    """Smeared central event: joining two pieces roughly doubles the lever arm, so the q/pT variance of the merged fit is
    well below that of the head alone; and chi2 per degree of freedom stays ~1 -- a rotation that moved the state off
    the track would cost chi2 of the order of (shift / 0.1 cm)^2 per hit."""
    ev = make_event(1, 1000)
    o = orc.track(ev)
    s, succ, pred, (par, cov, chi2, used, osec) = _merged(orc, ev, o)
    heads = np.nonzero((pred < 0) & (succ >= 0))[0]
    assert len(heads) > 2500
    ratio = cov[heads, 14] / o["refit_cov"][heads, 14]
    assert np.median(ratio) < 0.5
    ndf = 2 * used[heads] - 5
    ok = ndf > 40
    assert 0.85 < np.median(chi2[heads][ok] / ndf[ok]) < 1.15


def test_merged_refit_handmade_line_through_two_sectors(orc):
    """A straight line (Bz = 0) with hits placed by plane geometry in sector 1 (rows 20..39) and sector 2 (rows 40..59):
    every residual is zero in the right frames, so the fit returns the line exactly and uses all 40 hits."""
    n_rows = 80
    xr = 85.0 + (160.0 / 151.0) * np.arange(n_rows)
    p0, d = np.array([70.0, 38.0]), np.deg2rad(48.0)
    az = lambda sct: np.deg2rad((sct % 18 + 0.5) * 20.0)      # noqa: E731

    def local_hit(sct, row):
        ca, sa = np.cos(az(sct)), np.sin(az(sct))
        px, py = p0[0] * ca + p0[1] * sa, -p0[0] * sa + p0[1] * ca
        phi = d - az(sct)
        t = (xr[row] - px) / np.cos(phi)
        return py + t * np.sin(phi), 3.0 + 0.25 * t, phi

    ys, zs, counts = [], [], np.zeros(36 * n_rows, dtype=np.int64)
    for sct, rows in ((1, range(20, 40)), (2, range(40, 60))):
        for r in rows:
            yy, zz, _ = local_hit(sct, r)
            ys.append(yy)
            zs.append(zz)
            counts[sct * n_rows + r] += 1
    ro = np.concatenate([[0], np.cumsum(counts)]).astype(np.uint32)
    y, z = np.array(ys), np.array(zs)
    off, cnt, ids = np.array([0, 20], np.int32), np.array([20, 20], np.int32), np.arange(40, dtype=np.int32)
    succ, pred = np.array([1, -1], np.int32), np.array([-1, 0], np.int32)
    par, cov, chi2, used, osec = orc.refit_merged(y, z, ro, 36, n_rows, xr, 0.0, off, cnt, ids, succ, pred)
    y0, z0, phi0 = local_hit(1, 20)
    assert used.tolist() == [40, 0] and osec[0] == 1 and par[0, 0] == xr[20]
    assert abs(par[0, 1] - y0) < 1e-9 and abs(par[0, 2] - z0) < 1e-9
    assert abs(par[0, 3] - np.sin(phi0)) < 1e-11 and abs(par[0, 4] - 0.25) < 1e-11 and chi2[0] < 1e-16
    # the other direction of rotation: the same line entered as sector 2 -> sector 1 must NOT fit (wrong frames)
    ys2 = [local_hit(2, r)[0] for r in range(20, 40)] + [local_hit(1, r)[0] for r in range(40, 60)]
    par2, _, chi2_2, used2, _ = orc.refit_merged(np.array(ys2), z, ro, 36, n_rows, xr, 0.0, off, cnt, ids, succ, pred)
    assert chi2_2[0] > 1e3 or used2[0] < 40
