"""Seeded synthetic TPC events shaped like BASELINE.json configs[0..4].

Stand-in for the paper's workloads (ALICE 50 kHz Pb-Pb MC and 2022/2023 raw data),
which are not available.  Recipe: SURVEY.md section 8(d) and Appendix D, restated in DESIGN.md.

Everything here is written in *global helix* terms (circle of radius R around a centre, arc length from
the origin) and is independent of the tracker's sector-local (y, z, sin phi, tan lambda, q/pT)
parametrisation: it contains none of the method's arithmetic (no transport, no filter, no windows).

Output of make_event(): an Event with
    y, z          int32[N]   fixed-point cluster coordinates, units_per_cm = 640, grouped by (sector, row)
    row_offsets   uint32[n_sectors*n_rows + 1]  CSR over (sector, row)
    label         int64[N]   track_id*64 + piece, or -1 for noise
    y_exact, z_exact float64[N]  un-smeared, un-quantised crossing (NaN for noise)   [test pins only]
    truth         dict of per-track arrays (pt, eta, phi0, q, t0_us, side)
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

from .rng import Rng

UNITS_PER_CM = 640.0
N_ROWS = 152
X_FIRST, X_LAST = 85.0, 245.0
TAN10 = float(np.tan(np.deg2rad(10.0)))
C_LIGHT = 0.00299792458  # GeV/(T cm)
V_DRIFT = 2.58  # cm/us
Z_MAX_TRUE = 250.0


def row_x(n_rows: int = N_ROWS) -> np.ndarray:
    return X_FIRST + np.arange(n_rows, dtype=np.float64) * ((X_LAST - X_FIRST) / (n_rows - 1))


@dataclass
class Config:
    name: str
    n_sectors: int = 36
    open_sector: bool = False       # config 0: no +-10 deg cut, eta folded to >= 0
    collisions: int = 1
    tracks_per_collision: int = 4000
    mult_mode: str = "fixed"        # "fixed" | "exp" (mean tracks_per_collision, cap mult_cap)
    mult_cap: int = 4000
    time_mode: str = "zero"         # "zero" | "poisson50khz" | "uniform100us" | "window100us"
    pt_min: float = 0.1
    pt_slope: float = 0.5
    looper_frac: float = 0.0        # fraction of tracks with pT uniform in [0.05, 0.2]
    all_legs: bool = False          # follow returning legs / up to 5 turns (config 4)
    sigma_y: float = 0.1
    sigma_z: float = 0.15
    noise: float = 0.05
    bz: float = 0.5
    n_rows: int = N_ROWS
    row_pitches: tuple = ()         # ((n_gaps, pitch_cm), ...) from row 0 at x = 85 cm; empty = equidistant 85..245 cm


CONFIGS = {
    0: Config("cfg0_single_sector_100trk", n_sectors=1, open_sector=True, tracks_per_collision=100,
              pt_min=0.2, noise=0.0),
    1: Config("cfg1_central_PbPb_4000trk"),
    2: Config("cfg2_50kHz_PbPb_100coll", collisions=100, tracks_per_collision=1200, mult_mode="exp",
              time_mode="poisson50khz"),
    3: Config("cfg3_pp_pileup_5000coll", collisions=5000, tracks_per_collision=30, pt_slope=0.4,
              time_mode="uniform100us", noise=0.02),
    # 3b: the "about 2M clusters" reading of config 3
    30: Config("cfg3b_pp_pileup_500coll", collisions=500, tracks_per_collision=30, pt_slope=0.4,
               time_mode="uniform100us", noise=0.02),
    4: Config("cfg4_stress_loopers", tracks_per_collision=3000, looper_frac=0.4, all_legs=True,
              sigma_y=0.2, sigma_z=0.3, noise=0.2),
}


@dataclass
class Event:
    cfg: Config
    seed: int
    n_sectors: int
    n_rows: int
    row_x: np.ndarray
    y: np.ndarray
    z: np.ndarray
    row_offsets: np.ndarray
    label: np.ndarray
    y_exact: np.ndarray
    z_exact: np.ndarray
    truth: dict = field(default_factory=dict)
    z_extent_cm: float = Z_MAX_TRUE

    @property
    def n(self) -> int:
        return int(self.y.shape[0])

    def sector_row(self) -> tuple[np.ndarray, np.ndarray]:
        """(sector, row) of every cluster, from the CSR offsets."""
        counts = np.diff(self.row_offsets.astype(np.int64))
        sr = np.repeat(np.arange(counts.size), counts)
        return sr // self.n_rows, sr % self.n_rows


def _draw_collisions(cfg: Config, rng: Rng):
    nc = cfg.collisions
    if cfg.mult_mode == "fixed":
        mult = np.full(nc, cfg.tracks_per_collision, dtype=np.int64)
    else:
        m = rng.exponential(11, nc, float(cfg.tracks_per_collision))
        mult = np.minimum(np.floor(m).astype(np.int64), cfg.mult_cap)
    if cfg.time_mode == "zero":
        t0 = np.zeros(nc)
    elif cfg.time_mode == "poisson50khz":      # SURVEY P39 reading (b): exponential gaps, mean 20 us
        t0 = np.cumsum(rng.exponential(12, nc, 20.0))
        t0 -= t0[0]
    elif cfg.time_mode == "window100us":       # SURVEY P39 reading (a): all inside one drift window
        t0 = rng.uniform(12, nc) * 100.0
    elif cfg.time_mode == "uniform100us":
        t0 = rng.uniform(12, nc) * 100.0
    else:
        raise ValueError(cfg.time_mode)
    return mult, t0


def _crossings(cfg: Config, xr: np.ndarray, pt, eta, phi0, q, alphas):
    """Row-plane crossings of global helices from the origin.

    Returns flat arrays (track_local_index, sector_azimuth_index, row, y_local, z_true, piece).
    Global helix, arc length s >= 0, sense of rotation h = -q (Appendix D):
        psi(s) = psi0 + h s / R  (direction angle in the sector frame),  x'(s) = (R/h)(sin psi - sin psi0),
        y'(s) = -(R/h)(cos psi - cos psi0),  Z(s) = s sinh(eta).
    """
    R = pt / (C_LIGHT * cfg.bz)                      # (T,)
    h = -q                                           # (T,)
    psi0 = phi0[:, None] - alphas[None, :]           # (T,S)
    psi0 = (psi0 + np.pi) % (2 * np.pi) - np.pi
    A = np.sin(psi0)[:, :, None] + (h / R)[:, None, None] * xr[None, None, :]   # (T,S,R)
    ok = np.abs(A) <= 1.0
    base = np.arcsin(np.clip(A, -1.0, 1.0))
    two_pi = 2 * np.pi
    if cfg.all_legs:
        branches = (base, np.pi - base)
        extra = range(5)
        max_turn = 5 * two_pi
    else:
        branches = (base,)
        extra = range(1)
        max_turn = np.pi
    out = []
    hh = h[:, None, None]
    RR = R[:, None, None]
    p0 = psi0[:, :, None]
    sh = np.sinh(eta)[:, None, None]
    ymax = xr[None, None, :] * TAN10
    for b in branches:
        turn0 = ((b - p0) * hh) % two_pi
        for m in extra:
            turn = turn0 + two_pi * m
            psi = p0 + hh * turn
            s = turn * RR
            yl = -(RR / hh) * (np.cos(psi) - np.cos(p0))
            zt = s * sh
            good = ok & (turn > 0) & (turn <= max_turn) & (np.abs(zt) <= Z_MAX_TRUE)
            if not cfg.open_sector:
                good &= np.abs(yl) <= ymax
            ti, si, ri = np.nonzero(good)
            if ti.size == 0:
                continue
            ps = psi[ti, si, ri]
            p00 = psi0[ti, si]
            piece = np.abs(np.floor((ps - np.pi / 2) / np.pi) - np.floor((p00 - np.pi / 2) / np.pi)).astype(np.int64)
            out.append((ti, si, ri, yl[ti, si, ri], zt[ti, si, ri], piece))
    if not out:
        z = np.zeros(0, dtype=np.int64)
        return z, z, z, np.zeros(0), np.zeros(0), z
    return tuple(np.concatenate([o[i] for o in out]) for i in range(6))


def make_event(cfg_id: int | Config, seed: int | None = None, *, sigma_scale: float = 1.0,
               noise: float | None = None, n_tracks: int | None = None, collisions: int | None = None,
               time_mode: str | None = None, chunk: int = 1500) -> Event:
    """Generate one event.  seed defaults to 1000*cfg_id.  Keyword knobs are for pins:
    sigma_scale=0 gives exact helices (still quantised in y/z; y_exact/z_exact hold the doubles)."""
    if isinstance(cfg_id, Config):
        cfg, cid = cfg_id, 99
    else:
        cfg, cid = CONFIGS[cfg_id], int(cfg_id)
    if seed is None:
        seed = 1000 * cid
    cfg = Config(**{**cfg.__dict__})
    if noise is not None:
        cfg.noise = noise
    if n_tracks is not None:
        cfg.tracks_per_collision = n_tracks
    if collisions is not None:
        cfg.collisions = collisions
    if time_mode is not None:
        cfg.time_mode = time_mode
    rng = Rng(seed)
    if cfg.row_pitches:             # pad rows in regions of different pitch (NEXT-4, P48)
        gaps = np.concatenate([np.full(k, float(p)) for k, p in cfg.row_pitches])
        assert gaps.size == cfg.n_rows - 1
        xr = X_FIRST + np.concatenate([[0.0], np.cumsum(gaps)])
    else:
        xr = row_x(cfg.n_rows)
    n_az = 1 if cfg.n_sectors == 1 else 18
    alphas = np.zeros(1) if n_az == 1 else (np.arange(18) + 0.5) * np.deg2rad(20.0)

    mult, t0c = _draw_collisions(cfg, rng)
    nt = int(mult.sum())
    coll_of = np.repeat(np.arange(mult.size), mult)
    pt = cfg.pt_min + rng.exponential(21, nt, cfg.pt_slope)
    if cfg.looper_frac > 0:
        is_loop = rng.uniform(26, nt) < cfg.looper_frac
        pt = np.where(is_loop, 0.05 + 0.15 * rng.uniform(27, nt), pt)
    eta = -0.9 + 1.8 * rng.uniform(22, nt)
    if cfg.open_sector:
        eta = np.abs(eta)
        phi0 = (-1.0 + 2.0 * rng.uniform(23, nt)) * np.deg2rad(10.0)
    else:
        phi0 = 2 * np.pi * rng.uniform(23, nt)
    q = np.where(rng.uniform(24, nt) < 0.5, -1.0, 1.0)
    t0 = t0c[coll_of]
    side = (eta < 0).astype(np.int64)            # 0 = A side (z >= 0), 1 = C side

    trk, sec, row, yl, zt = [], [], [], [], []
    piece = []
    for a in range(0, nt, chunk):
        b = min(nt, a + chunk)
        ti, si, ri, y_, z_, pc = _crossings(cfg, xr, pt[a:b], eta[a:b], phi0[a:b], q[a:b], alphas)
        trk.append(ti + a)
        sec.append(si + n_az * side[ti + a] if cfg.n_sectors > 1 else si)
        row.append(ri)
        yl.append(y_)
        zt.append(z_)
        piece.append(pc)
    trk = np.concatenate(trk) if trk else np.zeros(0, dtype=np.int64)
    sec = np.concatenate(sec) if sec else np.zeros(0, dtype=np.int64)
    row = np.concatenate(row) if row else np.zeros(0, dtype=np.int64)
    yl = np.concatenate(yl) if yl else np.zeros(0)
    zt = np.concatenate(zt) if zt else np.zeros(0)
    piece = np.concatenate(piece) if piece else np.zeros(0, dtype=np.int64)

    sgn = np.where(side[trk] == 0, 1.0, -1.0)
    z_meas = zt + sgn * t0[trk] * V_DRIFT         # drift-time shift away from z = 0 on each side
    ns = trk.size
    y_sm = yl + sigma_scale * cfg.sigma_y * rng.normal(31, ns)
    z_sm = z_meas + sigma_scale * cfg.sigma_z * rng.normal(32, ns)
    label = trk * 64 + np.minimum(piece, 63)

    n_sr = cfg.n_sectors * cfg.n_rows
    sr = sec * cfg.n_rows + row
    z_ext = Z_MAX_TRUE + float(t0c.max()) * V_DRIFT
    if cfg.noise > 0:
        sig_count = np.bincount(sr, minlength=n_sr).astype(np.float64)
        n_noise = rng.poisson(41, cfg.noise * sig_count)
        nn = int(n_noise.sum())
        nsr = np.repeat(np.arange(n_sr), n_noise)
        nrow = nsr % cfg.n_rows
        nsec = nsr // cfg.n_rows
        ny = (-1.0 + 2.0 * rng.uniform(42, nn)) * xr[nrow] * TAN10
        nz = rng.uniform(43, nn) * z_ext * np.where(nsec < 18, 1.0, -1.0)
        sr = np.concatenate([sr, nsr])
        y_sm = np.concatenate([y_sm, ny])
        z_sm = np.concatenate([z_sm, nz])
        label = np.concatenate([label, np.full(nn, -1, dtype=np.int64)])
        yl = np.concatenate([yl, np.full(nn, np.nan)])
        z_meas = np.concatenate([z_meas, np.full(nn, np.nan)])

    n = sr.size
    # group by (sector,row); order inside a row is a seeded shuffle
    order = np.lexsort((rng.permutation_keys(51, n), sr))
    sr = sr[order]
    yi = np.rint(y_sm[order] * UNITS_PER_CM).astype(np.int32)
    zi = np.rint(z_sm[order] * UNITS_PER_CM).astype(np.int32)
    offs = np.zeros(n_sr + 1, dtype=np.uint32)
    offs[1:] = np.cumsum(np.bincount(sr, minlength=n_sr))
    truth = dict(pt=pt, eta=eta, phi0=phi0, q=q, t0_us=t0, side=side,
                 alphas=alphas, n_az=n_az)
    return Event(cfg=cfg, seed=seed, n_sectors=cfg.n_sectors, n_rows=cfg.n_rows, row_x=xr,
                 y=yi, z=zi, row_offsets=offs, label=label[order],
                 y_exact=yl[order], z_exact=z_meas[order], truth=truth, z_extent_cm=z_ext)


def truth_params_at(ev: Event, track: int, sector: int, x: float):
    """Truth (y, z, sin phi, tan lambda, q/pT) of `track`'s outgoing leg at local x of `sector`,
    from the global-helix expressions of Appendix D (used only by test pins)."""
    t = ev.truth
    R = t["pt"][track] / (C_LIGHT * ev.cfg.bz)
    h = -t["q"][track]
    alpha = t["alphas"][sector % t["n_az"]]
    psi0 = (t["phi0"][track] - alpha + np.pi) % (2 * np.pi) - np.pi
    A = np.sin(psi0) + h * x / R
    psi = np.arcsin(A)
    turn = ((psi - psi0) * h) % (2 * np.pi)
    s = turn * R
    y = -(R / h) * (np.cos(psi0 + h * turn) - np.cos(psi0))
    sgn = 1.0 if t["side"][track] == 0 else -1.0
    z = s * np.sinh(t["eta"][track]) + sgn * t["t0_us"][track] * V_DRIFT
    return np.array([y, z, A, np.sinh(t["eta"][track]), t["q"][track] / t["pt"][track]])


def concat_events(events: list[Event]) -> Event:
    """Stack events as extra sectors (the tracker treats sectors as independent units, so a batch of B
    events is one input with B*n_sectors sectors).  Labels are offset so they stay unique."""
    e0 = events[0]
    ys, zs, labs, yex, zex, offs = [], [], [], [], [], [np.zeros(1, dtype=np.int64)]
    base = 0
    lab_base = 0
    for e in events:
        ys.append(e.y)
        zs.append(e.z)
        lab = e.label.copy()
        lab[lab >= 0] += lab_base * 64
        labs.append(lab)
        yex.append(e.y_exact)
        zex.append(e.z_exact)
        offs.append(e.row_offsets[1:].astype(np.int64) + base)
        base += e.n
        lab_base += int(e.truth["pt"].size)
    return Event(cfg=e0.cfg, seed=e0.seed, n_sectors=e0.n_sectors * len(events), n_rows=e0.n_rows, row_x=e0.row_x,
                 y=np.concatenate(ys), z=np.concatenate(zs),
                 row_offsets=np.concatenate(offs).astype(np.uint32), label=np.concatenate(labs),
                 y_exact=np.concatenate(yex), z_exact=np.concatenate(zex), truth={},
                 z_extent_cm=max(e.z_extent_cm for e in events))
