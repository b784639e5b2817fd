"""Pins for the oracle's integer stages (neighbours, cleaner, chains, seeds) -- SURVEY 8(c) pin table.
None of these retype the oracle's loops: they use hand-made cases with answers worked out by hand,
invariants, and the brute-force == pruned equality north_star asks for."""
import numpy as np
import pytest

from gen.events import make_event
from gen.rng import Rng


def _rows(rows):
    """rows: list over rows of list of (y, z) -> (y, z, row_offsets) for one sector."""
    y = np.array([p[0] for r in rows for p in r], dtype=np.int32)
    z = np.array([p[1] for r in rows for p in r], dtype=np.int32)
    off = np.zeros(len(rows) + 1, dtype=np.uint32)
    off[1:] = np.cumsum([len(r) for r in rows])
    return y, z, off


def test_handmade_straight_line_beats_kink(orc):
    # row0: ids 0,1   row1: id 2   row2: ids 3,4
    # cluster 2 at (0,0); down candidates (-100,-50) id0 and (300,0) id1; up candidates (100,50) id3, (90,40) id4
    y, z, off = _rows([[(-100, -50), (300, 0)], [(0, 0)], [(100, 50), (90, 40)]])
    up, dn = orc.neighbours(y, z, off, 1, 3, brute=True)
    # (u=3,d=0): ddy = 100-100 = 0, ddz = 50-50 = 0 -> cost 0 is the minimum
    assert up.tolist() == [-1, -1, 3, -1, -1] and dn.tolist() == [-1, -1, 0, -1, -1]
    up2, dn2 = orc.neighbours(y, z, off, 1, 3, brute=False)
    assert np.array_equal(up, up2) and np.array_equal(dn, dn2)


def test_cost_value_and_cmax_boundary(orc):
    p = orc.default_params()
    # single pair: ddy = 10, ddz = 5 -> cost = 9*100 + 4*25 = 1000
    y, z, off = _rows([[(0, 0)], [(0, 0)], [(10, 5)]])
    p.c_max = 1000
    up, dn = orc.neighbours(y, z, off, 1, 3, p, brute=True)
    assert up[1] == 2 and dn[1] == 0
    p.c_max = 999
    up, dn = orc.neighbours(y, z, off, 1, 3, p, brute=True)
    assert up[1] == -1 and dn[1] == -1
    # default C_max = 16 * (9 * 6 * 64^2) = 3538944 : 2-dof chi2 of 16 at nominal smearing (P8, P10)
    assert orc.default_params().c_max == 16 * 9 * 6 * 64 * 64 == 3538944


def test_window_is_inclusive_and_centred_on_cluster(orc):
    p = orc.default_params()
    p.c_max = 2**31 - 1
    for (dy, dz, inside) in [(1280, 0, True), (1281, 0, False), (0, 1600, True), (0, -1601, False),
                             (-1280, -1600, True)]:
        y, z, off = _rows([[(0, 0)], [(0, 0)], [(dy, dz)]])
        up, dn = orc.neighbours(y, z, off, 1, 3, p, brute=True)
        assert (up[1] == 2) == inside, (dy, dz)
        up2, _ = orc.neighbours(y, z, off, 1, 3, p, brute=False)
        assert up2[1] == up[1]


def test_tie_break_lexicographic_ids(orc):
    # two up candidates mirror-symmetric in y about the straight continuation -> equal cost; smaller id wins (P9)
    y, z, off = _rows([[(0, 0)], [(0, 0)], [(7, 0), (-7, 0)]])
    up, dn = orc.neighbours(y, z, off, 1, 3, brute=True)
    assert up[1] == 2
    y, z, off = _rows([[(7, 0), (-7, 0)], [(0, 0)], [(0, 0)]])
    up, dn = orc.neighbours(y, z, off, 1, 3, brute=True)
    assert dn[2] == 0 and up[2] == 3


def test_first_and_last_row_have_no_links_and_no_cross_sector_links(orc):
    ev = make_event(1, n_tracks=300)
    up, dn = orc.neighbours(ev.y, ev.z, ev.row_offsets, ev.n_sectors, ev.n_rows)
    sec, row = ev.sector_row()
    assert np.all(up[(row == 0) | (row == ev.n_rows - 1)] == -1)
    assert np.all(dn[(row == 0) | (row == ev.n_rows - 1)] == -1)
    has = up >= 0
    assert np.all(dn[has] >= 0)                      # both or none
    assert np.all(sec[up[has]] == sec[has]) and np.all(row[up[has]] == row[has] + 1)
    assert np.all(sec[dn[has]] == sec[has]) and np.all(row[dn[has]] == row[has] - 1)


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_pruned_equals_bruteforce_on_dense_random(orc, seed):
    """north_star pin: grid neighbour search == brute-force all-pairs search on tiny inputs (dense, many ties)."""
    rng = Rng(seed)
    n_rows, per_row = 6, 60
    n = n_rows * per_row * 2
    y = (rng.uniform(1, n) * 6000 - 3000).astype(np.int32)
    z = (rng.uniform(2, n) * 8000 - 4000).astype(np.int32)
    y[::7] = (y[::7] // 64) * 64            # force exact cost ties
    z[::5] = (z[::5] // 64) * 64
    off = (np.arange(2 * n_rows + 1) * per_row).astype(np.uint32)
    a = orc.neighbours(y, z, off, 2, n_rows, brute=True)
    b = orc.neighbours(y, z, off, 2, n_rows, brute=False)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])
    assert (a[0] >= 0).sum() > 50


def test_pruned_equals_bruteforce_config0(orc):
    ev = make_event(0)
    a = orc.neighbours(ev.y, ev.z, ev.row_offsets, 1, ev.n_rows, brute=True)
    b = orc.neighbours(ev.y, ev.z, ev.row_offsets, 1, ev.n_rows, brute=False)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


def test_z_translation_invariance(orc):
    ev = make_event(0)
    a = orc.neighbours(ev.y, ev.z, ev.row_offsets, 1, ev.n_rows)
    b = orc.neighbours(ev.y, ev.z + np.int32(1234567), ev.row_offsets, 1, ev.n_rows)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


def test_permutation_invariance_of_links(orc):
    """Shuffling clusters inside each row (ids relabelled) gives the same links up to relabelling, where
    the winning pair is unique (exact cost ties are broken by id and may legitimately change)."""
    ev = make_event(0)
    rng = Rng(77)
    keys = rng.bits(1, ev.n)
    sr = np.repeat(np.arange(ev.n_rows), np.diff(ev.row_offsets.astype(np.int64)))
    perm = np.lexsort((keys, sr))               # new position j holds old cluster perm[j]
    inv = np.empty_like(perm)
    inv[perm] = np.arange(ev.n)
    up0, dn0 = orc.neighbours(ev.y, ev.z, ev.row_offsets, 1, ev.n_rows)
    up1, dn1 = orc.neighbours(ev.y[perm], ev.z[perm], ev.row_offsets, 1, ev.n_rows)
    # map new-id links back to old ids
    up1o = np.where(up1[inv] >= 0, perm[np.maximum(up1[inv], 0)], -1)
    dn1o = np.where(dn1[inv] >= 0, perm[np.maximum(dn1[inv], 0)], -1)
    same = (up0 == up1o) & (dn0 == dn1o)
    assert same.mean() > 0.999
    assert np.array_equal(up0 >= 0, up1o >= 0)


def test_cleaner_mutual_idempotent_and_handmade(orc):
    # hand-made: 0<->1 reciprocal; 2 points up to 1 but 1 points down to 0 -> 2's link is dropped
    up = np.array([1, -1, 1, -1], dtype=np.int32)
    dn = np.array([-1, 0, -1, -1], dtype=np.int32)
    upc, dnc = orc.clean_links(up, dn)
    assert upc.tolist() == [1, -1, -1, -1] and dnc.tolist() == [-1, 0, -1, -1]
    ev = make_event(4, n_tracks=300)
    up, dn = orc.neighbours(ev.y, ev.z, ev.row_offsets, ev.n_sectors, ev.n_rows)
    upc, dnc = orc.clean_links(up, dn)
    h = np.nonzero(upc >= 0)[0]
    assert np.array_equal(dnc[upc[h]], h)                    # mutual (north_star pin)
    h = np.nonzero(dnc >= 0)[0]
    assert np.array_equal(upc[dnc[h]], h)
    up2, dn2 = orc.clean_links(upc, dnc)
    assert np.array_equal(up2, upc) and np.array_equal(dn2, dnc)   # idempotent
    assert (upc >= 0).sum() < (up >= 0).sum()                # the stress config does drop links


def test_chains_partition_and_seed_rule(orc):
    ev = make_event(1, n_tracks=400)
    up, dn = orc.neighbours(ev.y, ev.z, ev.row_offsets, ev.n_sectors, ev.n_rows)
    upc, dnc = orc.clean_links(up, dn)
    p = orc.default_params()
    p.l_min = 1
    ss_all, sl_all = orc.find_seeds(upc, dnc, p)             # every chain with >= 2 clusters (start has an up link)
    isolated = ((upc < 0) & (dnc < 0)).sum()
    assert sl_all.sum() + isolated == ev.n                   # chains + isolated clusters partition the event
    assert np.all(np.diff(ss_all) > 0)                       # ascending start id (P14)
    # vertex-disjoint, monotone in row
    sec, row = ev.sector_row()
    seen = np.zeros(ev.n, dtype=bool)
    for s, l in zip(ss_all[:200], sl_all[:200]):
        c, k = s, 0
        while c >= 0:
            assert not seen[c]
            seen[c] = True
            if upc[c] >= 0:
                assert row[upc[c]] == row[c] + 1
            c = upc[c]
            k += 1
        assert k == l
    p.l_min = 5
    ss, sl = orc.find_seeds(upc, dnc, p)
    keep = sl_all >= 5
    assert np.array_equal(ss, ss_all[keep]) and np.array_equal(sl, sl_all[keep])


def test_zero_smearing_one_pure_chain_per_track(orc):
    ev = make_event(0, sigma_scale=0.0)
    up, dn = orc.neighbours(ev.y, ev.z, ev.row_offsets, 1, ev.n_rows)
    upc, dnc = orc.clean_links(up, dn)
    ss, sl = orc.find_seeds(upc, dnc)
    assert len(ss) == 100
    for s in ss:
        c, labs = s, set()
        while c >= 0:
            labs.add(int(ev.label[c]))
            c = upc[c]
        assert len(labs) == 1
    assert len({int(ev.label[s]) for s in ss}) == 100


# ---- NEXT-4 / P48: rows that are not equidistant (pitch-weighted straightness) ----
PADPLANE = ((62, 0.75), (33, 1.0), (29, 1.2), (27, 1.5))      # 152 rows in four regions of different pitch


def test_weighted_cost_prefers_the_straight_line_through_unequal_gaps(orc):
    """Row 0 -> row 1 is 1 cm, row 1 -> row 2 is 2 cm (weights 64, 128).  The straight continuation of d -> h lies twice
    as far from h as d does; the unweighted second difference would pick the mirror image of d instead."""
    w = np.array([64, 128], dtype=np.int32)
    y, z, off = _rows([[(-100, -50)], [(0, 0)], [(100, 50), (200, 100)]])      # ids: d = 0, h = 1, u = 2 (mirror), 3 (line)
    up, dn = orc.neighbours(y, z, off, 1, 3, brute=True, gap_w=w)
    assert up[1] == 3 and dn[1] == 0
    up0, _ = orc.neighbours(y, z, off, 1, 3, brute=True)
    assert up0[1] == 2                                          # what P8 for equal pitches gives on the same clusters
    up2, dn2 = orc.neighbours(y, z, off, 1, 3, brute=False, gap_w=w)
    assert up2[1] == 3 and dn2[1] == 0


def test_weighted_cost_value_and_threshold(orc):
    """D_y = wa y_u + wb y_d - (wa + wb) y_h = 64 * 10 = 640 -> cost = 9 * 640^2 = 3 686 400; accepted iff
    4 cost <= c_max (wa + wb)^2 = c_max * 36 864, i.e. iff c_max >= 400."""
    w = np.array([64, 128], dtype=np.int32)
    y, z, off = _rows([[(0, 0)], [(0, 0)], [(10, 0)]])
    p = orc.default_params()
    p.c_max = 400
    assert orc.neighbours(y, z, off, 1, 3, p, brute=True, gap_w=w)[0][1] == 2
    p.c_max = 399
    assert orc.neighbours(y, z, off, 1, 3, p, brute=True, gap_w=w)[0][1] == -1


def test_equal_weights_are_the_unweighted_reading(orc):
    ev = make_event(1, 9, n_tracks=300)
    a = orc.neighbours(ev.y, ev.z, ev.row_offsets, ev.n_sectors, ev.n_rows)
    b = orc.neighbours(ev.y, ev.z, ev.row_offsets, ev.n_sectors, ev.n_rows, gap_w=np.full(ev.n_rows - 1, 68, np.int32))
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])
    assert orc.pitch_weights(ev.row_x) is None                  # 160/151 cm everywhere -> one weight, 68


def _padplane_event(seed, **kw):
    from gen.events import Config
    cfg = Config("padplane_4_regions", n_sectors=36, tracks_per_collision=400, row_pitches=PADPLANE, **kw)
    return make_event(cfg, seed=seed)


def test_weighted_pruned_equals_bruteforce_on_a_four_region_geometry(orc):
    ev = _padplane_event(3)
    w = orc.pitch_weights(ev.row_x)
    assert w is not None and sorted(set(w.tolist())) == [48, 64, 77, 96]
    a = orc.neighbours(ev.y, ev.z, ev.row_offsets, ev.n_sectors, ev.n_rows, brute=True, gap_w=w)
    b = orc.neighbours(ev.y, ev.z, ev.row_offsets, ev.n_sectors, ev.n_rows, brute=False, gap_w=w)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


def test_exact_helices_on_unequal_pitches_give_one_pure_chain_per_track(orc):
    """The zero-smearing pin of the chain finder on the four-region geometry: with the weighted cost a helix stays
    'straight' across the pitch changes (rows 62, 95, 124), so no chain breaks there; with the unweighted cost the
    kink at a pitch change costs 9 * (0.25 * slope * 640)^2 and chains of inclined tracks break."""
    from gen.events import Config
    cfg = Config("padplane_open_sector", n_sectors=1, open_sector=True, tracks_per_collision=100, pt_min=0.2, noise=0.0,
                 row_pitches=PADPLANE)
    ev = make_event(cfg, seed=5, sigma_scale=0.0)
    w = orc.pitch_weights(ev.row_x)
    up, dn = orc.neighbours(ev.y, ev.z, ev.row_offsets, 1, ev.n_rows, gap_w=w)
    upc, dnc = orc.clean_links(up, dn)
    ss, sl = orc.find_seeds(upc, dnc)
    sec, row = ev.sector_row()
    n_tracks = len(set((ev.label[ev.label >= 0] // 64).tolist()))
    assert len(ss) == n_tracks
    for s0 in ss:                                               # every chain is one particle from end to end
        labs, c = [], s0
        while c >= 0:
            labs.append(ev.label[c] // 64)
            c = upc[c]
        assert len(set(labs)) == 1
    up0, dn0 = orc.neighbours(ev.y, ev.z, ev.row_offsets, 1, ev.n_rows)      # unweighted on the same clusters
    ss0, _ = orc.find_seeds(*orc.clean_links(up0, dn0))
    assert len(ss0) > n_tracks                                   # chains break at the pitch changes
