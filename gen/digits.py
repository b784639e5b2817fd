"""Seeded synthetic TPC digits (pad, time bin, ADC) for the clusterizer (NEXT-2, P53..P56).

Stand-in for the raw data of the paper's "Clustering" step, which is not available.  Every cluster of
a generated event (gen/events.py: its smeared double-precision position) deposits a charge on the pads and time bins
around it with a Gaussian pad and time response; deposits of neighbouring clusters add up; the sum is quantised to a
10-bit ADC and zero-suppressed.  No method arithmetic lives here: no peak finding, no centroid.

    pad p   <->  y = (p - (n_pads - 1) / 2) * pad_cm
    time t  <->  |z| = t * time_cm                (the sign of z is the sector's side)
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

from .rng import Rng

PAD_UNITS = 256          # pad pitch in fixed-point units: 0.4 cm
TIME_UNITS = 330         # time-bin width in fixed-point units: 0.515625 cm (0.2 us at 2.58 cm/us)
UNITS_PER_CM = 640.0


@dataclass
class Digits:
    n_sectors: int
    n_rows: int
    n_pads: int
    n_time: int
    pad: np.ndarray          # uint16 [n_digits]
    time: np.ndarray         # uint16 [n_digits]
    adc: np.ndarray          # uint16 [n_digits], 1..1023
    offsets: np.ndarray      # uint32 [n_sectors * n_rows + 1]; digits of a (sector,row) ascend by (time, pad)
    truth_sr: np.ndarray     # per generated cluster: sector * n_rows + row
    truth_y: np.ndarray      # its position in cm (doubles), as deposited
    truth_z: np.ndarray
    truth_q: np.ndarray      # its total charge in ADC counts

    @property
    def n(self) -> int:
        return int(self.pad.shape[0])


def make_digits(ev, seed: int | None = None, *, q_mean: float = 120.0, q_min: float = 30.0, sigma_pad: float = 0.55,
                sigma_time: float = 0.75, zero_suppression: int = 2, n_pads: int | None = None) -> Digits:
    """Digits for the clusters of `ev` (a gen.events.Event).  Charge per cluster = q_min + Exp(q_mean); response
    widths in pads / time bins; ADC values below `zero_suppression` are dropped, values above 1023 saturate."""
    rng = Rng(ev.seed * 7 + 13 if seed is None else seed)
    pad_cm, time_cm = PAD_UNITS / UNITS_PER_CM, TIME_UNITS / UNITS_PER_CM
    yc = ev.y / UNITS_PER_CM          # the event's (smeared, quantised) cluster positions in cm
    zc = np.abs(ev.z / UNITS_PER_CM)
    if n_pads is None:
        n_pads = int(np.ceil(2 * (np.abs(yc).max() + 3 * pad_cm) / pad_cm)) | 1      # odd: a pad sits at y = 0
    n_time = int(np.ceil((zc.max() + 4 * time_cm) / time_cm)) + 2
    n = ev.n
    sec, row = ev.sector_row()
    sr = sec * ev.n_rows + row
    q = q_min + rng.exponential(1, n, q_mean)
    pf = yc / pad_cm + (n_pads - 1) / 2.0            # fractional pad / time coordinates
    tf = zc / time_cm
    p0 = np.rint(pf).astype(np.int64)
    t0 = np.rint(tf).astype(np.int64)
    keys, vals = [], []
    norm = 1.0 / (2 * np.pi * sigma_pad * sigma_time)
    for dp in range(-2, 3):
        for dt in range(-3, 4):
            p, t = p0 + dp, t0 + dt
            ok = (p >= 0) & (p < n_pads) & (t >= 0) & (t < n_time)
            a = q * norm * np.exp(-0.5 * ((p - pf) / sigma_pad) ** 2 - 0.5 * ((t - tf) / sigma_time) ** 2)
            keys.append(((sr[ok] * n_time + t[ok]) * n_pads + p[ok]))
            vals.append(a[ok])
    keys = np.concatenate(keys)
    vals = np.concatenate(vals)
    uk, inv = np.unique(keys, return_inverse=True)            # ascending (sr, time, pad)
    summed = np.bincount(inv, weights=vals, minlength=uk.size)
    adc = np.minimum(np.floor(summed + 0.5 * rng.uniform(2, uk.size)), 1023).astype(np.int64)
    keep = adc >= zero_suppression
    uk, adc = uk[keep], adc[keep]
    d_sr = uk // (n_time * n_pads)
    rem = uk % (n_time * n_pads)
    n_sr = ev.n_sectors * ev.n_rows
    offsets = np.zeros(n_sr + 1, dtype=np.uint32)
    offsets[1:] = np.cumsum(np.bincount(d_sr, minlength=n_sr))
    return Digits(n_sectors=ev.n_sectors, n_rows=ev.n_rows, n_pads=n_pads, n_time=n_time,
                  pad=(rem % n_pads).astype(np.uint16), time=(rem // n_pads).astype(np.uint16), adc=adc.astype(np.uint16),
                  offsets=offsets, truth_sr=sr, truth_y=yc, truth_z=zc, truth_q=q)
