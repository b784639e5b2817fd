"""Pins for the oracle's NEXT-3 residual transform (readings P50..P52): worked-out predictor values,
exactness on lines and parabolas, the floor rule, lossless round trip, and the entropy a track model buys."""
import numpy as np

from gen.events import make_event


def _one_track(orc, rows, ys, zs, n_rows=32):
    """A single sector holding exactly the clusters of one track (one per listed row); returns its residual streams."""
    rows, ys, zs = np.asarray(rows), np.asarray(ys, np.int32), np.asarray(zs, np.int32)
    counts = np.zeros(n_rows, np.int64)
    counts[rows] = 1
    ro = np.concatenate([[0], np.cumsum(counts)]).astype(np.uint32)

    class Ev:
        pass

    ev = Ev()
    ev.n_rows, ev.n_sectors, ev.y, ev.z, ev.row_offsets = n_rows, 1, ys, zs, ro
    o = dict(trk_seed=np.array([0]), trk_hit_offset=np.array([0], np.int32), trk_n_owned=np.array([len(rows)], np.int32),
             hit_ids=np.arange(len(rows), dtype=np.int32))
    return orc.compress(ev, o), o


def test_headers_and_first_difference(orc):
    (drow, ry, rz), _ = _one_track(orc, [3, 4, 6], [100, 130, 190], [-7, -9, -13])
    assert drow.tolist() == [3, 1, 2]
    assert (ry[0], rz[0]) == (100, -7)                  # j = 0: absolute
    assert (ry[1], rz[1]) == (30, -2)                   # j = 1: first difference
    # j = 2: two-point line with gaps g1 = 1, g2 = 2: pred_y = 130 + floor(30 * 2 / 1) = 190, pred_z = -9 + (-2 * 2) = -13
    assert (ry[2], rz[2]) == (0, 0)


def test_two_point_predictor_uses_the_row_gaps_and_floors(orc):
    # rows 2, 5, 7: g1 = 3, g2 = 2; y: 10 -> 17 (slope 7/3 per row): pred = 17 + floor(7 * 2 / 3) = 17 + 4 = 21
    # z: 0 -> -7: pred = -7 + floor(-14 / 3) = -7 - 5 = -12   (floor, not truncation: -14/3 = -4.67 -> -5)
    (drow, ry, rz), _ = _one_track(orc, [2, 5, 7], [10, 17, 30], [0, -7, -20])
    assert drow.tolist() == [2, 3, 2] and ry[2] == 30 - 21 and rz[2] == -20 - (-12)


def test_four_point_predictor_value_and_its_conditions(orc):
    # consecutive rows 0..4, y = 0, 10, 20, 31, c4: pred = floor((2*31 + 20 - 0) / 2) = 41; odd numerator floors down
    (_, ry, rz), _ = _one_track(orc, [0, 1, 2, 3, 4], [0, 10, 20, 31, 50], [1, -1, 2, -2, 0])
    assert ry[4] == 50 - 41
    assert rz[4] == 0 - ((2 * -2 + 2 - 1) // 2)        # floor(-3 / 2) = -2
    assert ry[3] == 31 - (20 + 10) and ry[2] == 20 - 20        # j = 2, 3 have fewer than four predecessors: two-point line
    # a gap anywhere among the last five rows switches back to the two-point line
    (_, ry2, _), _ = _one_track(orc, [0, 1, 2, 4, 5], [0, 10, 20, 31, 50], [0] * 5)
    assert ry2[4] == 50 - (31 + (31 - 20) * 1 // 2)            # g1 = 2, g2 = 1: floor(11 / 2) = 5


def test_straight_lines_compress_to_zero_residuals(orc):
    rows = np.arange(2, 30)
    (drow, ry, rz), _ = _one_track(orc, rows, 50 + 7 * rows, -900 - 13 * rows)
    assert np.all(ry[2:] == 0) and np.all(rz[2:] == 0) and np.all(drow[1:] == 1)
    rows = np.array([1, 2, 4, 5, 9, 10, 11, 12, 13, 20])
    (drow, ry, rz), _ = _one_track(orc, rows, 6 * rows, 12 * rows)       # slope divisible by every gap: exact with gaps too
    assert np.all(ry[2:] == 0) and np.all(rz[2:] == 0)


def test_parabola_residual_is_the_textbook_extrapolation_error(orc):
    """y = a r^2: the two-point line misses the next point by 2a (second difference); the least-squares line through
    the last four points, extrapolated one row, misses it by 5a: sum_i w_i (r-i)^2 with w = (1, 1/2, 0, -1/2)."""
    a = 4
    rows = np.arange(0, 12)
    (_, ry, _), _ = _one_track(orc, rows, a * rows * rows, 0 * rows)
    assert ry[2] == 2 * a and ry[3] == 2 * a
    assert np.all(ry[4:] == 5 * a)


def test_round_trip_is_lossless(orc):
    ev = make_event(4, n_tracks=600)
    o = orc.track(ev)
    drow, ry, rz = orc.compress(ev, o)
    row, y, z = orc.decompress(o["trk_hit_offset"], o["trk_n_owned"], drow, ry, rz)
    sec, rw = ev.sector_row()
    h = o["hit_ids"]
    assert np.array_equal(row, rw[h]) and np.array_equal(y, ev.y[h]) and np.array_equal(z, ev.z[h])


def test_histogram_and_entropy(orc):
    off, cnt = np.array([0, 5], np.int32), np.array([5, 4], np.int32)
    res = np.array([9, 9, 0, 1, -1, 9, 9, 70000, -70000], np.int32)        # j >= 2: 0, 1, -1 | 70000, -70000
    hist = orc.residual_histogram(off, cnt, res, 2)
    assert hist.sum() == 5 and hist[32768] == 1 and hist[32769] == 1 and hist[32767] == 1
    assert hist[65535] == 1 and hist[0] == 1                                # clamped into the edge bins
    assert abs(orc.entropy_bits(hist) - np.log2(5)) < 1e-12
    assert orc.entropy_bits(np.array([8, 0, 0])) == 0.0 and abs(orc.entropy_bits(np.array([1, 1, 2])) - 1.5) < 1e-12


def test_track_model_saves_bits_on_a_central_event(orc):
    """What the transform buys on configs[1]: residual entropy per coordinate against the raw 32-bit words and against
    the first difference (no track model).  sigma_y = 64 units: an ideal predictor leaves log2(64 sqrt(2 pi e)) = 8.0
    bits; the four-point line leaves sqrt(2.5) more (+0.66 bit)."""
    ev = make_event(1, 1000, n_tracks=1500)
    o = orc.track(ev)
    drow, ry, rz = orc.compress(ev, o)
    hy = orc.entropy_bits(orc.residual_histogram(o["trk_hit_offset"], o["trk_n_owned"], ry, 2))
    hz = orc.entropy_bits(orc.residual_histogram(o["trk_hit_offset"], o["trk_n_owned"], rz, 2))
    # first differences of the same hits, for comparison
    h = o["hit_ids"]
    first = np.ones(len(h), bool)
    first[o["trk_hit_offset"]] = False
    dy = np.diff(ev.y[h], prepend=0)[first]
    hd = orc.entropy_bits(np.bincount(np.clip(dy + 32768, 0, 65535), minlength=65536))
    assert 8.0 < hy < 9.3 and 8.5 < hz < 9.9, (hy, hz)
    assert hd > hy + 1.0
    assert (drow[first] == 1).mean() > 0.97
