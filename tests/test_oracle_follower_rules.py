"""Hand-made pins for the *rules* of the oracle's follower and selection (SURVEY 8(c) "Stage 4", "Stage 5"):
the row search and its gate (P17, P21), the miss/stop logic of the extension phases (P20), the initial state (P19),
the final transport to the lowest hit (P23) and the tracklet-length filter on voters (P24).

Every expected value is worked out here from closed-form geometry, never from orc_*: the tracks are straight lines
(Bz = 0, so q/pT decouples) whose hits lie exactly on the line.  Then every residual is zero, the filter state stays
exactly on the line whatever the covariance is, and the predicted position in any row is the line itself.  For a line
along x (sin phi = tan lambda = 0) the y and z fits decouple into two textbook two-parameter line fits with a Gaussian
prior, whose prediction variance is [1, x] I^-1 [1, x]^T with I = prior information + sum of [1, x_i]^T [1, x_i] / sigma^2.
"""
import numpy as np
import pytest

PITCH = 160.0 / 151.0
N_ROWS = 30
ROW_X = 85.0 + PITCH * np.arange(N_ROWS)


class Sector:
    """One sector of hand-placed clusters; ids follow the CSR order (row by row, in the order added)."""

    def __init__(self, n_rows=N_ROWS, n_sectors=1):
        self.rows = [[] for _ in range(n_rows * n_sectors)]
        self.n_rows, self.n_sectors = n_rows, n_sectors

    def add(self, row, y, z, sector=0):
        self.rows[sector * self.n_rows + row].append((float(y), float(z)))
        return (row, len(self.rows[sector * self.n_rows + row]) - 1, sector)

    def build(self):
        off = np.zeros(len(self.rows) + 1, dtype=np.uint32)
        off[1:] = np.cumsum([len(r) for r in self.rows])
        y = np.array([p[0] for r in self.rows for p in r], dtype=np.float64)
        z = np.array([p[1] for r in self.rows for p in r], dtype=np.float64)
        return y, z, off

    def gid(self, handle, off):
        row, k, sector = handle
        return int(off[sector * self.n_rows + row]) + k


def follow(orc, sec, chain, params=None, bz=0.0, search_mode=0):
    """Runs orc_follow for one seed whose chain is the list of handles `chain` (consecutive rows)."""
    y, z, off = sec.build()
    ids = [sec.gid(h, off) for h in chain]
    upc = np.full(len(y), -1, dtype=np.int32)
    for a, b in zip(ids[:-1], ids[1:]):
        upc[a] = b
    par, cov, chi2, n_hits, hits = orc.follow(y, z, off, sec.n_sectors, sec.n_rows, ROW_X[:sec.n_rows], bz, upc,
                                              np.array([ids[0]], np.int32), np.array([len(ids)], np.int32), params,
                                              search_mode)
    return dict(par=par[0], cov=cov[0], chi2=chi2[0], n_hits=int(n_hits[0]), hits=hits[0], off=off, sec=sec)


def line_chain(sec, r_first, r_last, y_of=lambda x: 0.0, z_of=lambda x: 0.0):
    return [sec.add(r, y_of(ROW_X[r]), z_of(ROW_X[r])) for r in range(r_first, r_last + 1)]


def pred_var(prior_var_pos, prior_var_slope, sigma2, x_hits, x_pred):
    """Variance of a straight-line fit's prediction at x_pred: Gaussian prior on (position at x = 0, slope), hits at
    x_hits with variance sigma2.  Textbook weighted least squares in information form."""
    info = np.diag([1.0 / prior_var_pos, 1.0 / prior_var_slope])
    for x in x_hits:
        a = np.array([1.0, x])
        info += np.outer(a, a) / sigma2
    a = np.array([1.0, x_pred])
    return float(a @ np.linalg.solve(info, a))


MODES = [0, 1]   # full-row scan (the definition) and the oracle's z-sorted pruning


# ------------------------------------------------------------------------------------------------- P20, phase B
@pytest.mark.parametrize("mode", MODES)
def test_extension_up_survives_max_miss_minus_one_empty_rows_and_stops_after_max_miss(orc, mode):
    p = orc.default_params()
    assert p.max_miss == 5
    for gap, found in ((4, True), (5, False)):
        sec = Sector()
        chain = line_chain(sec, 2, 7)
        top = sec.add(8 + gap, 0.0, 0.0)          # rows 8 .. 8+gap-1 are empty
        r = follow(orc, sec, chain, search_mode=mode)
        assert (r["hits"][8 + gap] == sec.gid(top, r["off"])) == found, gap
        assert r["n_hits"] == 6 + (1 if found else 0)
        assert np.all(r["hits"][8:8 + gap] == -1)


@pytest.mark.parametrize("mode", MODES)
def test_miss_counter_resets_after_a_hit_going_up(orc, mode):
    sec = Sector()
    chain = line_chain(sec, 2, 7)
    a = sec.add(11, 0.0, 0.0)      # 3 empty rows (8, 9, 10), hit
    b = sec.add(15, 0.0, 0.0)      # 3 more empty rows (12, 13, 14), hit: 6 misses in total, never 5 in a row
    c = sec.add(21, 0.0, 0.0)      # 5 empty rows (16 .. 20): the extension stopped at row 20
    r = follow(orc, sec, chain, search_mode=mode)
    assert r["hits"][11] == sec.gid(a, r["off"]) and r["hits"][15] == sec.gid(b, r["off"])
    assert r["hits"][21] == -1 and r["n_hits"] == 8
    del c


@pytest.mark.parametrize("mode", MODES)
def test_extension_stops_at_the_last_row(orc, mode):
    sec = Sector()
    chain = line_chain(sec, N_ROWS - 8, N_ROWS - 3)
    top = sec.add(N_ROWS - 1, 0.0, 0.0)
    r = follow(orc, sec, chain, search_mode=mode)
    assert r["hits"][N_ROWS - 1] == sec.gid(top, r["off"]) and r["hits"][N_ROWS - 2] == -1


# ------------------------------------------------------------------------------------------------- P20, phase D
@pytest.mark.parametrize("mode", MODES)
def test_extension_down_stop_rule_and_counter_reset(orc, mode):
    for gap, found in ((4, True), (5, False)):
        sec = Sector()
        chain = line_chain(sec, 20, 25)
        low = sec.add(19 - gap, 0.0, 0.0)         # rows 19 .. 20-gap are empty
        r = follow(orc, sec, chain, search_mode=mode)
        assert (r["hits"][19 - gap] == sec.gid(low, r["off"])) == found, gap
    sec = Sector()
    chain = line_chain(sec, 20, 25)
    a = sec.add(16, 0.0, 0.0)      # rows 19, 18, 17 empty
    b = sec.add(12, 0.0, 0.0)      # rows 15, 14, 13 empty: found only if the counter was reset at row 16
    c = sec.add(6, 0.0, 0.0)       # rows 11 .. 7 empty: stop before row 6
    r = follow(orc, sec, chain, search_mode=mode)
    assert r["hits"][16] == sec.gid(a, r["off"]) and r["hits"][12] == sec.gid(b, r["off"]) and r["hits"][6] == -1
    assert r["n_hits"] == 8
    del c


@pytest.mark.parametrize("mode", MODES)
def test_rows_of_the_seed_without_a_hit_do_not_count_as_misses_on_the_way_down(orc, mode):
    """Phase C skips rows >= r0 that hold no recorded hit (SURVEY 8(c) Stage 4 Phase C): a 4-row hole in the upward
    extension plus 4 empty rows below the seed must not add up to a stop."""
    sec = Sector()
    chain = line_chain(sec, 10, 15)
    up = sec.add(20, 0.0, 0.0)       # rows 16 .. 19 empty on the way up
    dn = sec.add(5, 0.0, 0.0)        # rows 9 .. 6 empty on the way down
    r = follow(orc, sec, chain, search_mode=mode)
    assert r["hits"][20] == sec.gid(up, r["off"]) and r["hits"][5] == sec.gid(dn, r["off"])


# ------------------------------------------------------------------------------------------------- P21 gate, P17
def _first_row_above_chain_variances(p, n_chain):
    xs = PITCH * np.arange(n_chain)
    x_pred = PITCH * n_chain
    vy = pred_var(p.c_reset[0], p.c_reset[2], p.sigma_y ** 2, xs, x_pred)
    vz = pred_var(p.c_reset[1], p.c_reset[3], p.sigma_z ** 2, xs, x_pred)
    return vy, vz


@pytest.mark.parametrize("mode", MODES)
def test_gate_d_threshold_is_15_with_innovation_variances(orc, mode):
    """Candidate in the first row above a 6-hit chain at d = 15 (1 -+ 1e-6): accepted below, rejected above (P21:
    d < 15 strictly), with d = dy^2/(Cyy + sy^2) + dz^2/(Czz + sz^2) and Cyy, Czz the closed-form line-fit prediction
    variances.  Pins the threshold, the use of the *predicted* covariance and the + sigma^2 terms."""
    p = orc.default_params()
    vy, vz = _first_row_above_chain_variances(p, 6)
    sy2, sz2 = p.sigma_y ** 2, p.sigma_z ** 2
    assert 1e-3 < vy < 0.05 and 1e-3 < vz < 0.1          # sanity: well below the caps' scale
    for axis in ("y", "z", "both"):
        for scale, found in ((1 - 1e-6, True), (1 + 1e-6, False)):
            if axis == "y":
                dy, dz = np.sqrt(15.0 * (vy + sy2)) * scale, 0.0
            elif axis == "z":
                dy, dz = 0.0, np.sqrt(15.0 * (vz + sz2)) * scale
            else:
                dy, dz = np.sqrt(7.0 * (vy + sy2)) * scale, -np.sqrt(8.0 * (vz + sz2)) * scale
            assert abs(dy) < p.gate_y_cm and abs(dz) < p.gate_z_cm
            sec = Sector()
            chain = line_chain(sec, 3, 8)
            c = sec.add(9, dy, dz)
            r = follow(orc, sec, chain, search_mode=mode)
            assert (r["hits"][9] == sec.gid(c, r["off"])) == found, (axis, scale)


@pytest.mark.parametrize("mode", MODES)
def test_absolute_caps_2cm_and_2p5cm_inclusive(orc, mode):
    """P21: |dy| <= 2.0 cm and |dz| <= 2.5 cm restrict the candidates whatever d says (gate_d opened wide here)."""
    p = orc.default_params()
    p.gate_d = 1e9
    for dy, dz, found in ((2.0, 0.0, True), (2.0 + 1e-9, 0.0, False), (-2.0, 0.0, True), (0.0, 2.5, True),
                          (0.0, -2.5 - 1e-9, False), (2.0, -2.5, True), (1.0, 2.6, False)):
        sec = Sector()
        chain = line_chain(sec, 3, 8)
        c = sec.add(9, dy, dz)
        r = follow(orc, sec, chain, p, search_mode=mode)
        assert (r["hits"][9] == sec.gid(c, r["off"])) == found, (dy, dz)


@pytest.mark.parametrize("mode", MODES)
def test_nearest_candidate_uses_the_z_variance_for_the_z_term(orc, mode):
    """Two candidates: A off in z only, B off in y only, placed so that A is nearer with the definition's weights
    (1/(Czz + sz^2) on dz^2) and B would be nearer if the z term were weighted like the y term (P17)."""
    p = orc.default_params()
    vy, vz = _first_row_above_chain_variances(p, 6)
    wy, wz = 1.0 / (vy + p.sigma_y ** 2), 1.0 / (vz + p.sigma_z ** 2)
    dz_a = 0.30
    d_a = dz_a ** 2 * wz
    dy_b = np.sqrt(0.5 * (d_a + dz_a ** 2 * wy) / wy)     # d_A < d_B = dy_b^2 wy < dz_a^2 wy
    d_b = dy_b ** 2 * wy
    assert d_a < d_b < dz_a ** 2 * wy and d_b < 15
    for order in (0, 1):   # independent of which of the two has the smaller id
        sec = Sector()
        chain = line_chain(sec, 3, 8)
        if order == 0:
            a = sec.add(9, 0.0, dz_a)
            sec.add(9, dy_b, 0.0)
        else:
            sec.add(9, dy_b, 0.0)
            a = sec.add(9, 0.0, dz_a)
        r = follow(orc, sec, chain, search_mode=mode)
        assert r["hits"][9] == sec.gid(a, r["off"])


@pytest.mark.parametrize("mode", MODES)
def test_exact_distance_tie_goes_to_the_smaller_id(orc, mode):
    """Two candidates at (+1/8, -1/8) and (-1/8, +1/8) cm: identical d bit for bit; the smaller id wins (P17), also
    when the z-sorted scan meets the other one first."""
    for first_is_plus_z in (True, False):
        sec = Sector()
        chain = line_chain(sec, 3, 8)
        s = 1.0 if first_is_plus_z else -1.0
        a = sec.add(9, -0.125 * s, 0.125 * s)
        sec.add(9, 0.125 * s, -0.125 * s)
        r = follow(orc, sec, chain, search_mode=mode)
        assert r["hits"][9] == sec.gid(a, r["off"])


@pytest.mark.parametrize("mode", MODES)
def test_search_looks_only_at_the_seed_sector(orc, mode):
    sec = Sector(n_sectors=2)
    chain = line_chain(sec, 3, 8)
    sec.add(9, 0.0, 0.0, sector=1)          # perfect continuation, wrong sector (P33)
    r = follow(orc, sec, chain, search_mode=mode)
    assert r["hits"][9] == -1 and r["n_hits"] == 6


# ------------------------------------------------------------------------------------------------- P19, P23
def _sloped():
    y_of = lambda x: 3.0 + 0.75 * (x - ROW_X[0])            # noqa: E731   steep: dy = 0.79 cm per row
    z_of = lambda x: -20.0 + 0.9 * (x - ROW_X[0])           # noqa: E731
    return y_of, z_of


def test_initial_state_is_dy_over_chord_and_dz_over_chord(orc):
    """P19 on a steep straight line: sin phi = dy/chord and tan lambda = dz/chord (chord in the xy plane) are the exact
    line parameters, so every residual is zero and the fit returns the line to rounding.  With dz/dx, or dy/dx, the
    prior mean is off the line and the result moves by ~1e-3."""
    y_of, z_of = _sloped()
    sec = Sector()
    chain = [sec.add(r, y_of(ROW_X[r]), z_of(ROW_X[r])) for r in range(4, 14)]
    r = follow(orc, sec, chain)
    slope_y, slope_z = 0.75, 0.9
    norm = np.hypot(1.0, slope_y)
    assert r["par"][0] == ROW_X[4]
    assert abs(r["par"][1] - y_of(ROW_X[4])) < 1e-10 and abs(r["par"][2] - z_of(ROW_X[4])) < 1e-10
    assert abs(r["par"][3] - slope_y / norm) < 1e-11      # sin phi
    assert abs(r["par"][4] - slope_z / norm) < 1e-11      # tan lambda = dz / ds_xy
    assert r["par"][5] == 0.0 and r["chi2"] < 1e-18


@pytest.mark.parametrize("mode", MODES)
def test_final_state_is_transported_back_to_the_lowest_hit(orc, mode):
    """P23: Phase D runs 5 rows below the lowest hit before it stops; the reported state must be the line at the x of
    the lowest hit, not where the search stopped."""
    y_of, z_of = _sloped()
    sec = Sector()
    chain = [sec.add(r, y_of(ROW_X[r]), z_of(ROW_X[r])) for r in range(12, 20)]
    low = sec.add(10, y_of(ROW_X[10]), z_of(ROW_X[10]))       # row 11 empty, row 10 found, rows 9 .. 5 missed
    r = follow(orc, sec, chain, search_mode=mode)
    assert r["hits"][10] == sec.gid(low, r["off"]) and np.all(r["hits"][:10] == -1)
    assert r["par"][0] == ROW_X[10]
    assert abs(r["par"][1] - y_of(ROW_X[10])) < 1e-9 and abs(r["par"][2] - z_of(ROW_X[10])) < 1e-9
    # and when nothing is found below the seed, the lowest hit is the seed's first
    sec = Sector()
    chain = [sec.add(r, y_of(ROW_X[r]), z_of(ROW_X[r])) for r in range(12, 20)]
    r = follow(orc, sec, chain, search_mode=mode)
    assert r["par"][0] == ROW_X[12] and abs(r["par"][1] - y_of(ROW_X[12])) < 1e-9


def test_final_covariance_is_the_line_fit_covariance_at_the_lowest_hit(orc):
    """The reported covariance is the Phase C/D covariance transported to the lowest hit: for a line along x it is the
    textbook line-fit covariance with the P22 prior placed at the row where the upward pass ended."""
    p = orc.default_params()
    sec = Sector()
    chain = line_chain(sec, 12, 19)
    low = sec.add(10, 0.0, 0.0)
    r = follow(orc, sec, chain)
    # upward pass: chain to row 19, then 5 misses -> the reset happens at row 24; hits at rows 19..12 and 10
    x_top = ROW_X[24]
    xs = np.array([ROW_X[k] for k in list(range(12, 20)) + [10]]) - x_top
    vy = pred_var(p.c_reset[0], p.c_reset[2], p.sigma_y ** 2, xs, ROW_X[10] - x_top)
    vz = pred_var(p.c_reset[1], p.c_reset[3], p.sigma_z ** 2, xs, ROW_X[10] - x_top)
    assert abs(r["cov"][0] - vy) < 1e-9 * vy and abs(r["cov"][2] - vz) < 1e-9 * vz
    assert abs(r["cov"][14] - p.c_reset[4]) < 1e-12       # Bz = 0: q/pT never learns anything
    del low


# ------------------------------------------------------------------------------------------------- P24, P26
def test_short_tracklets_cast_no_vote(orc):
    """P24: a tracklet with fewer than n_min_tracklet (10) hits is discarded before the ownership contest: it owns
    nothing, not even clusters nobody else wants, and takes nothing from the survivor."""
    nr = 16
    hits = np.full((3, nr), -1, dtype=np.int32)
    hits[0, :9] = np.arange(0, 9)             # 9 hits: clusters 0..8 -> discarded
    hits[1, :12] = np.arange(5, 17)           # 12 hits: clusters 5..16
    hits[2, :10] = np.arange(20, 30)          # exactly 10 hits: survives
    n_hits = np.array([9, 12, 10], dtype=np.int32)
    owner, trk_seed, trk_n, trk_off, hit_ids = orc.select(30, nr, np.array([0, 5, 20], np.int32), n_hits, hits)
    assert owner[:5].tolist() == [-1] * 5
    assert owner[5:17].tolist() == [1] * 12 and owner[20:30].tolist() == [2] * 10
    assert trk_seed.tolist() == [1, 2] and trk_n.tolist() == [12, 10]
    # the discarded tracklet does not win ties either: same length as nobody, but a smaller start id than tracklet 1
    p = orc.default_params()
    p.n_min_tracklet = 13
    owner, trk_seed, *_ = orc.select(30, nr, np.array([0, 5, 20], np.int32), n_hits, hits, p)
    assert np.all(owner == -1) and len(trk_seed) == 0


def test_owned_count_threshold_is_separate_from_the_tracklet_threshold(orc):
    """P27: a surviving 12-hit tracklet that keeps only 9 of its hits is not output, but its votes still stand."""
    nr = 16
    hits = np.full((2, nr), -1, dtype=np.int32)
    hits[0, :12] = np.arange(0, 12)
    hits[1, :14] = np.concatenate([np.arange(9, 12), np.arange(12, 23)])   # takes 9, 10, 11 from tracklet 0
    n_hits = np.array([12, 14], dtype=np.int32)
    owner, trk_seed, trk_n, trk_off, hit_ids = orc.select(23, nr, np.array([0, 9], np.int32), n_hits, hits)
    assert owner[:9].tolist() == [0] * 9 and owner[9:].tolist() == [1] * 14
    assert trk_seed.tolist() == [1] and trk_n.tolist() == [14]
