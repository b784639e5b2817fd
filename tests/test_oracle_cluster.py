"""Pins for the oracle's NEXT-2 clusterizer (readings P53..P56): hand-made digit patterns with the centroid
worked out by hand, the plateau and threshold rules, overlapping blocks, the side sign, and position resolution against
the digit generator's truth."""
from types import SimpleNamespace

import numpy as np

from gen.digits import PAD_UNITS, TIME_UNITS, make_digits
from gen.events import make_event


def _digits(cells, n_pads=21, n_time=40, n_sectors=1, n_rows=2, sr=0):
    """cells: {(time, pad): adc} for one (sector,row) `sr`; everything else empty."""
    items = sorted(cells.items())
    off = np.zeros(n_sectors * n_rows + 1, np.uint32)
    off[sr + 1:] = len(items)
    return SimpleNamespace(n_sectors=n_sectors, n_rows=n_rows, n_pads=n_pads, n_time=n_time,
                           pad=np.array([k[1] for k, _ in items], np.uint16), time=np.array([k[0] for k, _ in items], np.uint16),
                           adc=np.array([v for _, v in items], np.uint16), offsets=off)


Y_OFF = (21 - 1) * PAD_UNITS // 2       # pad 10 is y = 0 with 21 pads


def test_single_symmetric_deposit_sits_on_its_pad_and_time_bin(orc):
    cells = {(10, 10): 100}
    for dt in (-1, 0, 1):
        for dp in (-1, 0, 1):
            if (dt, dp) != (0, 0):
                cells[(10 + dt, 10 + dp)] = 20
    c = orc.clusterize(_digits(cells))
    assert c["y"].tolist() == [10 * PAD_UNITS - Y_OFF] == [0] and c["z"].tolist() == [10 * TIME_UNITS]
    assert c["qtot"].tolist() == [260] and c["qmax"].tolist() == [100]
    assert c["row_offsets"].tolist() == [0, 1, 1]


def test_centroid_value_and_rounding(orc):
    """Peak 50 at (t, p) = (7, 4) with 30 on pad 5 and 10 on time bin 6: Q = 90, Sy = +30, St = -10.
    y = 4 * 256 - 2560 + rdiv(256 * 30, 90) = -1536 + round(85.33) = -1451;
    z = 7 * 330 + rdiv(330 * -10, 90) = 2310 + round(-36.67) = 2273."""
    c = orc.clusterize(_digits({(7, 4): 50, (7, 5): 30, (6, 4): 10}))
    assert c["y"].tolist() == [-1536 + 85] and c["z"].tolist() == [2310 - 37] and c["qtot"].tolist() == [90]
    # halves round up (towards +infinity): Sy / Q = 1/2 pad -> 128 exactly; -1/2 pad -> -128; 256 * 1 / 6 = 42.67 -> 43
    assert orc.clusterize(_digits({(7, 4): 30, (7, 5): 30}))["y"].tolist() == [-1536 + 128]
    assert orc.clusterize(_digits({(7, 4): 50, (7, 5): 10}))["y"].tolist() == [-1536 + 43]
    assert orc.clusterize(_digits({(7, 4): 25, (7, 5): 5, (7, 3): 10}), pad_units=3, time_units=330)["y"].tolist() == \
        [4 * 3 - (20 * 3) // 2 + 0]          # rdiv(3 * -5, 40) = floor((-30 + 40) / 80) = 0  (-0.375 rounds to 0)
    # 3 * 10 / 20 = 1.5 rounds up to 2 (plateau: the peak is the first cell, pad 3): y = 9 - 30 + 2
    assert orc.clusterize(_digits({(7, 4): 10, (7, 3): 10}), pad_units=3, time_units=330)["y"].tolist() == [-19]


def test_plateau_yields_its_first_cell_only(orc):
    """Two equal neighbouring maxima: the earlier one in (time, pad) order is >= the later one, the later one is not >
    the earlier one -> exactly one peak, the first."""
    c = orc.clusterize(_digits({(7, 4): 40, (7, 5): 40}))
    assert len(c["y"]) == 1 and c["y"][0] == 4 * PAD_UNITS - Y_OFF + 128 and c["qmax"][0] == 40
    c = orc.clusterize(_digits({(7, 4): 40, (8, 4): 40}))
    assert len(c["z"]) == 1 and c["z"][0] == 7 * TIME_UNITS + 165
    c = orc.clusterize(_digits({(7, 5): 40, (8, 4): 40}))      # diagonal neighbours: (7, 5) precedes (8, 4)
    assert len(c["z"]) == 1 and c["qtot"][0] == 80 and c["y"][0] == 5 * PAD_UNITS - Y_OFF - 128
    # a plateau whose first cell comes later in pad but earlier in time
    c = orc.clusterize(_digits({(7, 4): 10, (7, 3): 10}))
    assert len(c["y"]) == 1 and c["y"][0] == 3 * PAD_UNITS - Y_OFF + 128


def test_peak_threshold_and_strictness(orc):
    assert len(orc.clusterize(_digits({(7, 4): 5}))["y"]) == 0                  # below q_peak_min = 6
    assert len(orc.clusterize(_digits({(7, 4): 6}))["y"]) == 1
    assert len(orc.clusterize(_digits({(7, 4): 5}), q_peak_min=5)["y"]) == 1
    assert len(orc.clusterize(_digits({(7, 4): 50, (7, 5): 51}))["y"]) == 1      # 50 is not a peak next to 51
    assert orc.clusterize(_digits({(7, 4): 50, (7, 5): 51}))["qmax"].tolist() == [51]


def test_two_peaks_share_the_digits_between_them(orc):
    """Peaks at pads 4 and 6 of one time bin with a digit on pad 5: both are found, both blocks contain pad 5."""
    c = orc.clusterize(_digits({(7, 4): 60, (7, 5): 20, (7, 6): 50}))
    assert c["qtot"].tolist() == [80, 70] and c["qmax"].tolist() == [60, 50]
    assert c["y"].tolist() == [4 * PAD_UNITS - Y_OFF + 64, 6 * PAD_UNITS - Y_OFF - 73]      # 256*20/80 = 64; -256*20/70 = -73.1
    # order inside the row: ascending (time, pad) of the peak
    c = orc.clusterize(_digits({(9, 2): 30, (7, 15): 30, (7, 3): 30}))
    assert c["z"].tolist() == [7 * TIME_UNITS, 7 * TIME_UNITS, 9 * TIME_UNITS]
    assert c["y"].tolist() == [3 * PAD_UNITS - Y_OFF, 15 * PAD_UNITS - Y_OFF, 2 * PAD_UNITS - Y_OFF]


def test_edges_sides_and_rows(orc):
    c = orc.clusterize(_digits({(0, 0): 30, (0, 1): 10, (39, 20): 30}))       # corners of the (time, pad) plane
    assert c["y"].tolist() == [-Y_OFF + 64, 20 * PAD_UNITS - Y_OFF] and c["z"].tolist() == [0, 39 * TIME_UNITS]
    d = _digits({(7, 4): 50}, n_sectors=36, n_rows=3, sr=19 * 3 + 2)           # sector 19: C side
    c = orc.clusterize(d)
    assert c["z"].tolist() == [-7 * TIME_UNITS] and c["row_offsets"][19 * 3 + 2] == 0 and c["row_offsets"][19 * 3 + 3] == 1
    d = _digits({(7, 4): 50}, n_sectors=72, n_rows=3, sr=37 * 3)               # second event of a batch, A side again
    assert orc.clusterize(d)["z"].tolist() == [7 * TIME_UNITS]


def test_generated_clusters_come_back_at_their_positions(orc):
    """Against the generator's truth (independent code): on a sparse event almost every deposited cluster is found once,
    with a position error far below the pad and time-bin size."""
    ev = make_event(1, 5, n_tracks=150, noise=0.0)
    d = make_digits(ev)
    c = orc.clusterize(d)
    ro = c["row_offsets"].astype(np.int64)
    assert 0.97 * ev.n < len(c["y"]) < 1.02 * ev.n
    # match within each (sector,row) by nearest neighbour
    sr_found = np.repeat(np.arange(len(ro) - 1), np.diff(ro))
    side = np.where((d.truth_sr // ev.n_rows) // 18 % 2 == 1, -1.0, 1.0)
    ty, tz = d.truth_y * 640.0, d.truth_z * 640.0 * side
    order = np.argsort(d.truth_sr, kind="stable")
    starts = np.searchsorted(d.truth_sr[order], np.arange(len(ro)))
    dy, dz = [], []
    for sr in np.unique(sr_found)[:400]:
        t_idx = order[starts[sr]:starts[sr + 1]]
        f = slice(ro[sr], ro[sr + 1])
        for k in t_idx:
            dist = np.hypot(c["y"][f] - ty[k], c["z"][f] - tz[k])
            j = dist.argmin()
            if dist[j] < 200:
                dy.append(c["y"][f][j] - ty[k])
                dz.append(c["z"][f][j] - tz[k])
    dy, dz = np.array(dy), np.array(dz)
    assert len(dy) > 1000
    assert abs(dy.mean()) < 3 and abs(dz.mean()) < 4                    # unbiased (units of 1/640 cm)
    assert dy.std() < 0.12 * PAD_UNITS and dz.std() < 0.12 * TIME_UNITS   # ~0.04 cm and ~0.05 cm
