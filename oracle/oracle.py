"""ctypes loader + stage-by-stage driver for the CPU oracle (oracle/tpc_oracle.cpp).

TEST INFRASTRUCTURE, NOT PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this.  It never imports paper_2502_09138_b200.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import time

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libtpc_oracle.so")
_SRC = [os.path.join(_HERE, "tpc_oracle.cpp"), os.path.join(_HERE, "tpc_oracle.h")]


class Params(C.Structure):
    _fields_ = [
        ("w_y", C.c_int32), ("w_z", C.c_int32), ("cost_wy", C.c_int32), ("cost_wz", C.c_int32),
        ("c_max", C.c_int32), ("l_min", C.c_int32),
        ("units_per_cm", C.c_double), ("sigma_y", C.c_double), ("sigma_z", C.c_double),
        ("sinphi_max", C.c_double), ("max_miss", C.c_int32), ("n_min_tracklet", C.c_int32),
        ("gate_d", C.c_double), ("gate_y_cm", C.c_double), ("gate_z_cm", C.c_double),
        ("c_reset", C.c_double * 5), ("cq_per_tesla", C.c_double), ("n_min_owned", C.c_int32),
    ]


def build(force: bool = False) -> str:
    """Compile the oracle with g++ -O2 -fopenmp if missing or stale."""
    stale = (not os.path.exists(_SO)) or any(os.path.getmtime(s) > os.path.getmtime(_SO) for s in _SRC)
    if force or stale:
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-Wall",
                               _SRC[0], "-o", _SO])
    return _SO


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_find_seeds.restype = C.c_int64
        _lib.orc_select.restype = C.c_int64
        _lib.orc_update.restype = C.c_double
        _lib.orc_transport.restype = C.c_int
        _lib.orc_num_threads.restype = C.c_int
        _lib.orc_rotate.restype = C.c_int
        _lib.orc_match_chi2.restype = C.c_double
        _lib.orc_merge.restype = C.c_int64
        _lib.orc_clusterize.restype = C.c_int64
    return _lib


def default_params() -> Params:
    p = Params()
    lib().orc_default_params(C.byref(p))
    return p


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t))


def _i32(a):
    return _p(a, C.c_int32)


def _u32(a):
    return _p(a, C.c_uint32)


def _f64(a):
    return _p(a, C.c_double)


def pitch_weights(row_x):
    """P48: integer weight of every gap between consecutive rows, nearbyint(64 * pitch in cm); None when all weights
    are equal (then the cost is the plain second difference of P8)."""
    w = np.rint(64.0 * np.diff(np.asarray(row_x, dtype=np.float64))).astype(np.int32)
    return None if np.all(w == w[0]) else np.ascontiguousarray(w)


def neighbours(y, z, row_offsets, n_sectors, n_rows, params=None, brute=False, gap_w=None):
    p = params or default_params()
    n = y.shape[0]
    up = np.empty(n, dtype=np.int32)
    dn = np.empty(n, dtype=np.int32)
    f = lib().orc_neighbours_brute_w if brute else lib().orc_neighbours_pruned_w
    f(C.byref(p), C.c_int32(n_sectors), C.c_int32(n_rows), _i32(gap_w) if gap_w is not None else None, _i32(y), _i32(z),
      _u32(row_offsets), _i32(up), _i32(dn))
    return up, dn


def clean_links(up, dn):
    n = up.shape[0]
    upc = np.empty(n, dtype=np.int32)
    dnc = np.empty(n, dtype=np.int32)
    lib().orc_clean_links(C.c_int64(n), _i32(up), _i32(dn), _i32(upc), _i32(dnc))
    return upc, dnc


def find_seeds(upc, dnc, params=None):
    p = params or default_params()
    n = upc.shape[0]
    cap = n // max(1, p.l_min) + 1
    start = np.empty(cap, dtype=np.int32)
    length = np.empty(cap, dtype=np.int32)
    ns = lib().orc_find_seeds(C.byref(p), C.c_int64(n), _i32(upc), _i32(dnc), _i32(start), _i32(length))
    return start[:ns].copy(), length[:ns].copy()


def transport(state, cov, dx, cq, sinphi_max=0.95):
    st = np.array(state, dtype=np.float64)
    cv = None if cov is None else np.array(cov, dtype=np.float64).reshape(25)
    ok = lib().orc_transport(C.c_double(cq), C.c_double(sinphi_max), C.c_double(dx), _f64(st),
                             _f64(cv) if cv is not None else None)
    return bool(ok), st, (None if cv is None else cv.reshape(5, 5))


def jacobian(state, dx, cq):
    st = np.array(state, dtype=np.float64)
    F = np.empty(25, dtype=np.float64)
    lib().orc_jacobian(C.c_double(cq), C.c_double(dx), _f64(st), _f64(F))
    return F.reshape(5, 5)


def update(state, cov, ym, zm, sy2, sz2):
    st = np.array(state, dtype=np.float64)
    cv = np.array(cov, dtype=np.float64).reshape(25)
    chi2 = lib().orc_update(_f64(st), _f64(cv), C.c_double(ym), C.c_double(zm), C.c_double(sy2), C.c_double(sz2))
    return st, cv.reshape(5, 5), float(chi2)


def follow(y_cm, z_cm, row_offsets, n_sectors, n_rows, row_x, bz, upc, seed_start, seed_len, params=None,
           search_mode=1):
    p = params or default_params()
    ns = seed_start.shape[0]
    par = np.zeros((ns, 6), dtype=np.float64)
    cov = np.zeros((ns, 15), dtype=np.float64)
    chi2 = np.zeros(ns, dtype=np.float64)
    n_hits = np.zeros(ns, dtype=np.int32)
    hits = np.full((ns, n_rows), -1, dtype=np.int32)
    y_cm = np.ascontiguousarray(y_cm, dtype=np.float64)
    z_cm = np.ascontiguousarray(z_cm, dtype=np.float64)
    row_x = np.ascontiguousarray(row_x, dtype=np.float64)
    lib().orc_follow(C.byref(p), C.c_double(bz), C.c_int32(n_sectors), C.c_int32(n_rows), _f64(row_x), _f64(y_cm),
                     _f64(z_cm), _u32(row_offsets), _i32(upc), C.c_int64(ns), _i32(seed_start), _i32(seed_len),
                     C.c_int(search_mode), _f64(par), _f64(cov), _f64(chi2), _i32(n_hits), _i32(hits))
    return par, cov, chi2, n_hits, hits


def select(n, n_rows, seed_start, n_hits, hits, params=None):
    p = params or default_params()
    ns = seed_start.shape[0]
    owner = np.empty(n, dtype=np.int32)
    trk_seed = np.empty(ns, dtype=np.int32)
    trk_n = np.empty(ns, dtype=np.int32)
    trk_off = np.empty(ns, dtype=np.int32)
    hit_ids = np.empty(int(np.maximum(n_hits, 0).sum()) + 1, dtype=np.int32)
    nh = C.c_int64(0)
    hits = np.ascontiguousarray(hits, dtype=np.int32)
    nt = lib().orc_select(C.byref(p), C.c_int64(n), C.c_int32(n_rows), C.c_int64(ns), _i32(seed_start), _i32(n_hits),
                          _i32(hits), _i32(owner), _i32(trk_seed), _i32(trk_n), _i32(trk_off), _i32(hit_ids),
                          C.byref(nh))
    return owner, trk_seed[:nt].copy(), trk_n[:nt].copy(), trk_off[:nt].copy(), hit_ids[:nh.value].copy()


def refit(y_cm, z_cm, row_offsets, n_sectors, n_rows, row_x, bz, trk_hit_offset, trk_n_owned, hit_ids, params=None):
    """orc_refit: NEXT-1, refit of every output track over its owned hits (reading P41)."""
    p = params or default_params()
    nt = trk_n_owned.shape[0]
    par = np.zeros((nt, 6), dtype=np.float64)
    cov = np.zeros((nt, 15), dtype=np.float64)
    chi2 = np.zeros(nt, dtype=np.float64)
    n_used = np.zeros(nt, dtype=np.int32)
    y_cm = np.ascontiguousarray(y_cm, dtype=np.float64)
    z_cm = np.ascontiguousarray(z_cm, dtype=np.float64)
    row_x = np.ascontiguousarray(row_x, dtype=np.float64)
    lib().orc_refit(C.byref(p), C.c_double(bz), C.c_int32(n_sectors), C.c_int32(n_rows), _f64(row_x), _f64(y_cm),
                    _f64(z_cm), _u32(row_offsets), C.c_int64(nt), _i32(np.ascontiguousarray(trk_hit_offset, np.int32)),
                    _i32(np.ascontiguousarray(trk_n_owned, np.int32)), _i32(np.ascontiguousarray(hit_ids, np.int32)),
                    _f64(par), _f64(cov), _f64(chi2), _i32(n_used))
    return par, cov, chi2, n_used


MERGE_GAP_MAX = 25        # P43: rows between the last hit of a segment and the first hit of its continuation
MERGE_CHI2_MAX = 50.0     # P44: 5-parameter chi2 of the extrapolated state against the continuation's state


def rotate(x, state, cov, alpha, cq, sinphi_max=0.95):
    """orc_rotate: (ok, x', state', cov') in the frame turned by alpha."""
    xx = C.c_double(float(x))
    st = np.array(state, dtype=np.float64)
    cv = None if cov is None else np.array(cov, dtype=np.float64).reshape(25)
    ok = lib().orc_rotate(C.c_double(cq), C.c_double(sinphi_max), C.c_double(alpha), C.byref(xx), _f64(st),
                          _f64(cv) if cv is not None else None)
    return bool(ok), xx.value, st, (None if cv is None else cv.reshape(5, 5))


def match_chi2(par_a, cov_a, par_b, cov_b, alpha, cq, sinphi_max=0.95):
    pa, ca = np.ascontiguousarray(par_a, np.float64), np.ascontiguousarray(cov_a, np.float64)
    pb, cb = np.ascontiguousarray(par_b, np.float64), np.ascontiguousarray(cov_b, np.float64)
    return float(lib().orc_match_chi2(C.c_double(cq), C.c_double(sinphi_max), C.c_double(alpha), _f64(pa), _f64(ca),
                                      _f64(pb), _f64(cb)))


def merge(par, cov, sector, first_row, last_row, bz, params=None, n_per_side=18, sector_angle=np.deg2rad(20.0),
          gap_max=MERGE_GAP_MAX, chi2_max=MERGE_CHI2_MAX):
    """orc_merge over track records (par [nt, 6], cov [nt, 15]); returns (succ, pred, link_chi2, n_links)."""
    p = params or default_params()
    nt = int(np.asarray(sector).shape[0])
    par = np.ascontiguousarray(par, np.float64).reshape(nt, 6)
    cov = np.ascontiguousarray(cov, np.float64).reshape(nt, 15)
    sector = np.ascontiguousarray(sector, np.int32)
    first_row = np.ascontiguousarray(first_row, np.int32)
    last_row = np.ascontiguousarray(last_row, np.int32)
    succ = np.full(nt, -1, np.int32)
    pred = np.full(nt, -1, np.int32)
    chi2 = np.full(nt, -1.0, np.float64)
    nl = lib().orc_merge(C.c_double(p.cq_per_tesla * bz), C.c_double(p.sinphi_max), C.c_int32(n_per_side),
                         C.c_double(sector_angle), C.c_int32(gap_max), C.c_double(chi2_max), C.c_int64(nt), _f64(par),
                         _f64(cov), _i32(sector), _i32(first_row), _i32(last_row), _i32(succ), _i32(pred), _f64(chi2))
    return succ, pred, chi2, int(nl)


def refit_merged(y_cm, z_cm, row_offsets, n_sectors, n_rows, row_x, bz, trk_hit_offset, trk_n_owned, hit_ids, succ, pred,
                 params=None, n_per_side=18, sector_angle=np.deg2rad(20.0)):
    """orc_refit_merged (P47): refit over the hits of every chain of linked tracks; heads only (n_used > 0)."""
    p = params or default_params()
    nt = trk_n_owned.shape[0]
    par = np.zeros((nt, 6), dtype=np.float64)
    cov = np.zeros((nt, 15), dtype=np.float64)
    chi2 = np.zeros(nt, dtype=np.float64)
    n_used = np.zeros(nt, dtype=np.int32)
    out_sector = np.full(nt, -1, dtype=np.int32)
    lib().orc_refit_merged(C.byref(p), C.c_double(bz), C.c_int32(n_sectors), C.c_int32(n_rows),
                           _f64(np.ascontiguousarray(row_x, np.float64)), _f64(np.ascontiguousarray(y_cm, np.float64)),
                           _f64(np.ascontiguousarray(z_cm, np.float64)), _u32(row_offsets), C.c_int32(n_per_side),
                           C.c_double(sector_angle), C.c_int64(nt), _i32(np.ascontiguousarray(trk_hit_offset, np.int32)),
                           _i32(np.ascontiguousarray(trk_n_owned, np.int32)), _i32(np.ascontiguousarray(hit_ids, np.int32)),
                           _i32(np.ascontiguousarray(succ, np.int32)), _i32(np.ascontiguousarray(pred, np.int32)),
                           _f64(par), _f64(cov), _f64(chi2), _i32(n_used), _i32(out_sector))
    return par, cov, chi2, n_used, out_sector


def compress(ev, o):
    """orc_compress on the oracle's output tracks: (drow uint8, ry int32, rz int32) in hit-list order (P50)."""
    nh = len(o["hit_ids"])
    drow = np.zeros(max(nh, 1), np.uint8)
    ry = np.zeros(max(nh, 1), np.int32)
    rz = np.zeros(max(nh, 1), np.int32)
    lib().orc_compress(C.c_int32(ev.n_rows), _i32(ev.y), _i32(ev.z), _u32(ev.row_offsets),
                       C.c_int64(ev.n_sectors * ev.n_rows), C.c_int64(len(o["trk_seed"])),
                       _i32(np.ascontiguousarray(o["trk_hit_offset"], np.int32)),
                       _i32(np.ascontiguousarray(o["trk_n_owned"], np.int32)),
                       _i32(np.ascontiguousarray(o["hit_ids"], np.int32)), _p(drow, C.c_uint8), _i32(ry), _i32(rz))
    return drow[:nh], ry[:nh], rz[:nh]


def decompress(trk_hit_offset, trk_n_owned, drow, ry, rz):
    """orc_decompress: (row, y, z) of every hit from the residual streams (P51)."""
    nh = int(len(drow))
    row = np.zeros(max(nh, 1), np.int32)
    y = np.zeros(max(nh, 1), np.int32)
    z = np.zeros(max(nh, 1), np.int32)
    lib().orc_decompress(C.c_int64(len(trk_n_owned)), _i32(np.ascontiguousarray(trk_hit_offset, np.int32)),
                         _i32(np.ascontiguousarray(trk_n_owned, np.int32)),
                         _p(np.ascontiguousarray(drow, np.uint8), C.c_uint8), _i32(np.ascontiguousarray(ry, np.int32)),
                         _i32(np.ascontiguousarray(rz, np.int32)), _i32(row), _i32(y), _i32(z))
    return row[:nh], y[:nh], z[:nh]


def residual_histogram(trk_hit_offset, trk_n_owned, res, j_min=2):
    hist = np.zeros(65536, np.int64)
    lib().orc_residual_histogram(C.c_int64(len(trk_n_owned)), _i32(np.ascontiguousarray(trk_hit_offset, np.int32)),
                                 _i32(np.ascontiguousarray(trk_n_owned, np.int32)),
                                 _i32(np.ascontiguousarray(res, np.int32)), C.c_int32(j_min), _p(hist, C.c_int64))
    return hist


def rans_symbol(v, alphabet_bits):
    return int(lib().orc_rans_symbol(C.c_int32(int(v)), C.c_int32(alphabet_bits)))


def rans_normalise(counts):
    """P58: normalised frequencies (sum 65536) of a histogram over the alphabet."""
    counts = np.ascontiguousarray(counts, np.int64)
    freq = np.zeros(len(counts), np.uint32)
    lib().orc_rans_normalise(C.c_int32(len(counts)), _p(counts, C.c_int64), _u32(freq))
    return freq


def rans_encode(values, alphabet_bits=12, chunk=512):
    """P57..P60: dict(freq, chunk_off, esc_off, payload, escapes) of an int32 stream."""
    values = np.ascontiguousarray(values, np.int32)
    n = int(len(values))
    n_chunks = (n + chunk - 1) // chunk
    freq = np.zeros(1 << alphabet_bits, np.uint32)
    chunk_off = np.zeros(n_chunks + 1, np.uint32)
    esc_off = np.zeros(n_chunks + 1, np.uint32)
    payload = np.zeros(max(n_chunks * 4 + 2 * n, 1), np.uint8)
    escapes = np.zeros(max(n, 1), np.int32)
    lib().orc_rans_encode.restype = C.c_int64
    nbytes = lib().orc_rans_encode(_i32(values), C.c_int64(n), C.c_int32(alphabet_bits), C.c_int32(chunk), _u32(freq),
                                   _u32(chunk_off), _u32(esc_off), _p(payload, C.c_uint8), _i32(escapes))
    return dict(n=n, alphabet_bits=alphabet_bits, chunk=chunk, freq=freq, chunk_off=chunk_off, esc_off=esc_off,
                payload=payload[:nbytes].copy(), escapes=escapes[:int(esc_off[-1])].copy())


def rans_decode(enc):
    """The inverse of rans_encode."""
    n = enc["n"]
    values = np.zeros(max(n, 1), np.int32)
    payload = np.ascontiguousarray(np.concatenate([enc["payload"], np.zeros(2, np.uint8)]))
    escapes = np.ascontiguousarray(np.concatenate([enc["escapes"], np.zeros(1, np.int32)]))
    lib().orc_rans_decode(C.c_int64(n), C.c_int32(enc["alphabet_bits"]), C.c_int32(enc["chunk"]),
                          _u32(np.ascontiguousarray(enc["freq"], np.uint32)),
                          _u32(np.ascontiguousarray(enc["chunk_off"], np.uint32)),
                          _u32(np.ascontiguousarray(enc["esc_off"], np.uint32)), _p(payload, C.c_uint8), _i32(escapes),
                          _i32(values))
    return values[:n]


def entropy_bits(hist):
    """Empirical entropy in bits per symbol of a histogram: what an ideal entropy coder (the paper's rANS stage) needs."""
    h = np.asarray(hist, dtype=np.float64)
    n = h.sum()
    if n == 0:
        return 0.0
    p = h[h > 0] / n
    return float(-(p * np.log2(p)).sum())


CLUSTER_Q_PEAK_MIN = 6     # P53: smallest ADC value of a peak


def clusterize(d, n_per_side=18, pad_units=256, time_units=330, q_peak_min=CLUSTER_Q_PEAK_MIN):
    """orc_clusterize on gen.digits.Digits (duck-typed: n_sectors, n_rows, n_pads, n_time, pad, time, adc, offsets).
    Returns dict(y, z, qtot, qmax, row_offsets)."""
    cap = max(int(d.pad.shape[0]), 1)
    y = np.zeros(cap, np.int32)
    z = np.zeros(cap, np.int32)
    qt = np.zeros(cap, np.int32)
    qm = np.zeros(cap, np.int32)
    ro = np.zeros(d.n_sectors * d.n_rows + 1, np.uint32)
    u16 = lambda a: _p(np.ascontiguousarray(a, np.uint16), C.c_uint16)      # noqa: E731
    nc = lib().orc_clusterize(C.c_int32(d.n_sectors), C.c_int32(d.n_rows), C.c_int32(n_per_side), C.c_int32(d.n_pads),
                              C.c_int32(d.n_time), C.c_int32(pad_units), C.c_int32(time_units), C.c_int32(q_peak_min),
                              u16(d.pad), u16(d.time), u16(d.adc), _u32(np.ascontiguousarray(d.offsets, np.uint32)),
                              _i32(y), _i32(z), _i32(qt), _i32(qm), _u32(ro))
    return dict(y=y[:nc].copy(), z=z[:nc].copy(), qtot=qt[:nc].copy(), qmax=qm[:nc].copy(), row_offsets=ro)


def track_records(ev, o):
    """(sector, first_row, last_row) of the oracle's output tracks, from their owned hit lists."""
    sec, row = ev.sector_row()
    nt = len(o["trk_seed"])
    s = np.zeros(nt, np.int32)
    f = np.zeros(nt, np.int32)
    l = np.zeros(nt, np.int32)
    for t in range(nt):
        h = o["hit_ids"][o["trk_hit_offset"][t]: o["trk_hit_offset"][t] + o["trk_n_owned"][t]]
        s[t], f[t], l[t] = sec[h[0]], row[h[0]], row[h[-1]]
    return s, f, l


def track(ev, params=None, *, brute=False, search_mode=1, exact_coords=False, timings=None):
    """Whole path on one generated event (gen.events.Event).  Returns a dict with every stage's output.

    exact_coords=True feeds the follower the un-smeared, un-quantised doubles (y_exact/z_exact) instead of
    int/units_per_cm: the oracle-internal entry that bypasses quantisation (SURVEY 8c pin table)."""
    p = params or default_params()
    t = [time.perf_counter()]
    up, dn = neighbours(ev.y, ev.z, ev.row_offsets, ev.n_sectors, ev.n_rows, p, brute=brute,
                        gap_w=pitch_weights(ev.row_x))
    t.append(time.perf_counter())
    upc, dnc = clean_links(up, dn)
    ss, sl = find_seeds(upc, dnc, p)
    t.append(time.perf_counter())
    if exact_coords:
        y_cm, z_cm = ev.y_exact, ev.z_exact
    else:
        y_cm, z_cm = ev.y / p.units_per_cm, ev.z / p.units_per_cm
    par, cov, chi2, n_hits, hits = follow(y_cm, z_cm, ev.row_offsets, ev.n_sectors, ev.n_rows, ev.row_x, ev.cfg.bz,
                                          upc, ss, sl, p, search_mode)
    t.append(time.perf_counter())
    owner, trk_seed, trk_n, trk_off, hit_ids = select(ev.n, ev.n_rows, ss, n_hits, hits, p)
    t.append(time.perf_counter())
    rf_par, rf_cov, rf_chi2, rf_used = refit(y_cm, z_cm, ev.row_offsets, ev.n_sectors, ev.n_rows, ev.row_x, ev.cfg.bz,
                                             trk_off, trk_n, hit_ids, p)
    if timings is not None:
        timings.update(neighbours=t[1] - t[0], clean_seeds=t[2] - t[1], follow=t[3] - t[2], select=t[4] - t[3],
                       total=t[4] - t[0])
    return dict(link_up=up, link_dn=dn, up_c=upc, dn_c=dnc, seed_start=ss, seed_len=sl, par=par, cov=cov,
                chi2=chi2, n_hits=n_hits, hits=hits, owner=owner, trk_seed=trk_seed, trk_n_owned=trk_n,
                trk_hit_offset=trk_off, hit_ids=hit_ids, refit_par=rf_par, refit_cov=rf_cov, refit_chi2=rf_chi2,
                refit_used=rf_used)


def num_threads() -> int:
    return int(lib().orc_num_threads())
