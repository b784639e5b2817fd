"""Generator checks: determinism, sizes (BASELINE.json configs), and that clusters lie on the global helix."""
import numpy as np
import pytest

from gen.events import C_LIGHT, CONFIGS, make_event, row_x, truth_params_at


def test_deterministic_and_seed_dependent():
    a, b, c = make_event(0), make_event(0), make_event(0, seed=1)
    assert np.array_equal(a.y, b.y) and np.array_equal(a.z, b.z) and np.array_equal(a.row_offsets, b.row_offsets)
    assert a.n != c.n or not np.array_equal(a.y, c.y)


def test_sizes_match_baseline_configs():
    e0 = make_event(0)
    assert 12000 < e0.n < 16000 and e0.n_sectors == 1          # "about 15k clusters"
    e1 = make_event(1)
    assert 570_000 < e1.n < 640_000 and e1.n_sectors == 36     # "about 600k"
    assert 0.04 < (e1.label < 0).mean() < 0.055                # 5 % noise per row, relative to signal
    assert e1.row_offsets[-1] == e1.n and e1.row_offsets.size == 36 * 152 + 1
    rx = row_x()
    assert rx[0] == 85.0 and abs(rx[-1] - 245.0) < 1e-12 and np.allclose(np.diff(rx), 160.0 / 151)


def test_clusters_lie_on_circle_through_origin():
    """Independent of the crossing formula: transform the exact local crossing back to the global frame and
    check its distance to the helix centre equals R, and z = arc length * sinh(eta)."""
    ev = make_event(1, sigma_scale=0.0, noise=0.0, n_tracks=200)
    sec, row = ev.sector_row()
    t = ev.truth
    trk = ev.label // 64
    alpha = t["alphas"][sec % 18]
    xg = ev.row_x[row] * np.cos(alpha) - ev.y_exact * np.sin(alpha)
    yg = ev.row_x[row] * np.sin(alpha) + ev.y_exact * np.cos(alpha)
    R = t["pt"][trk] / (C_LIGHT * 0.5)
    h = -t["q"][trk]
    cx = -(R / h) * np.sin(t["phi0"][trk])
    cy = (R / h) * np.cos(t["phi0"][trk])
    assert np.max(np.abs(np.hypot(xg - cx, yg - cy) - R)) < 1e-8
    # arc length from the origin along the circle: s = R * (angle subtended at the centre), outgoing leg <= pi
    a0 = np.arctan2(0 - cy, 0 - cx)
    a1 = np.arctan2(yg - cy, xg - cx)
    s = R * (((a1 - a0) * h) % (2 * np.pi))
    assert np.max(np.abs(ev.z_exact - s * np.sinh(t["eta"][trk]))) < 1e-7
    # quantisation: int = rint(cm * 640)
    assert np.array_equal(ev.y, np.rint(ev.y_exact * 640).astype(np.int32))
    # A side <-> eta > 0
    assert np.all((sec < 18) == (t["eta"][trk] > 0))


def test_curvature_sign_positive_charge_bends_to_minus_y():
    """F = q v x B with B along +z: a positive particle moving along +x is deflected towards -y."""
    ev = make_event(0, sigma_scale=0.0)
    t = ev.truth
    k = int(np.argmax(t["q"] > 0))
    p0, p1 = truth_params_at(ev, k, 0, 100.0), truth_params_at(ev, k, 0, 200.0)
    assert p1[2] < p0[2]          # sin(phi) decreases with x for q > 0, Bz > 0
    assert p0[4] > 0


@pytest.mark.parametrize("cfg", [4, 30])
def test_other_configs_generate(cfg):
    ev = make_event(cfg, n_tracks=300 if cfg == 4 else None, collisions=20 if cfg == 30 else None)
    assert ev.n > 0 and ev.row_offsets[-1] == ev.n
    cnt = np.diff(ev.row_offsets.astype(np.int64))
    assert cnt.min() >= 0
    if cfg == 4:
        assert (ev.label[ev.label >= 0] % 64).max() >= 1     # returning legs present
        assert CONFIGS[4].sigma_y == 0.2
