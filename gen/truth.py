"""Truth matching of output tracks against generator labels (harness, not library).

Applied identically to the oracle's and the CUDA path's outputs; contains none of the method's arithmetic.
"""
from __future__ import annotations

import numpy as np


def match_tracks(ev, trk_sector, trk_hit_offset, trk_n_hits, hit_ids, purity=0.8, findable_min=30):
    """P30.  Output track matched to label l iff l >= 0 is the majority label of its hits with fraction
    >= purity, else fake.  Findable = (sector, label) with >= findable_min clusters.  Returns a dict with
    efficiency, fake_rate, clone_rate and counts."""
    lab = ev.label
    sec, _ = ev.sector_row()
    key = sec.astype(np.int64) * (1 << 40) + lab
    sig = lab >= 0
    uk, cnt = np.unique(key[sig], return_counts=True)
    findable = set(uk[cnt >= findable_min].tolist())
    n_out = len(trk_n_hits)
    matched = {}
    fakes = 0
    for t in range(n_out):
        ids = hit_ids[trk_hit_offset[t]: trk_hit_offset[t] + trk_n_hits[t]]
        l = lab[ids]
        vals, c = np.unique(l, return_counts=True)
        j = int(np.argmax(c))
        if vals[j] >= 0 and c[j] >= purity * len(ids):
            k = int(trk_sector[t]) * (1 << 40) + int(vals[j])
            matched[k] = matched.get(k, 0) + 1
        else:
            fakes += 1
    found = sum(1 for k in findable if k in matched)
    clones = sum(v - 1 for v in matched.values())
    return dict(n_out=n_out, n_findable=len(findable), n_found=found, n_fake=fakes, n_clone=clones,
                efficiency=found / max(1, len(findable)), fake_rate=fakes / max(1, n_out),
                clone_rate=clones / max(1, n_out))


def assignment_match(seed_a, off_a, n_a, hits_a, seed_b, off_b, n_b, hits_b):
    """P31.  Tracks keyed by seed start cluster id; a match = present in both with identical hit-id lists.
    Returns (fraction over max(n_a, n_b), list of matched (index_a, index_b))."""
    ib = {int(s): i for i, s in enumerate(seed_b)}
    pairs = []
    for i, s in enumerate(seed_a):
        j = ib.get(int(s))
        if j is None or n_a[i] != n_b[j]:
            continue
        if np.array_equal(hits_a[off_a[i]: off_a[i] + n_a[i]], hits_b[off_b[j]: off_b[j] + n_b[j]]):
            pairs.append((i, j))
    denom = max(len(seed_a), len(seed_b), 1)
    return len(pairs) / denom, pairs
