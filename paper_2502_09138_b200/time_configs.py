"""Per-stage device times of one tpc_track call on the synthetic configs of BASELINE.json (one event each).

    python -m paper_2502_09138_b200.time_configs 0 1 4 30 2 3      (30 = configs[3] at its stated size, 500 collisions)

Prints one line per config: clusters, seeds, output tracks, ms per call, clusters/s, the five stage times
(tpc_get_stage_ms_mean over five calls after three warm-up calls) and the grid the call chose.  bench.py is the
throughput benchmark (configs[1], batched); this is the table for the other workloads.
"""
from __future__ import annotations

import sys


def main(argv):
    import torch
    from gen.events import make_event
    from . import Tracker
    from .events import geometry_from_event, upload

    for cfg in [int(a) for a in argv] or [0, 1, 4, 30]:
        ev = make_event(cfg)
        trk = Tracker(geometry_from_event(ev))
        y, z, ro = upload(ev)
        out = trk.alloc_out(ev.n, track_capacity=ev.n // 20 + 1024, hit_capacity=ev.n + 1024)
        for _ in range(3):
            trk.track(y, z, ro, out)
        torch.cuda.synchronize()
        trk.set_stage_timing(True)
        for _ in range(5):
            trk.track(y, z, ro, out)
        torch.cuda.synchronize()
        st, _ = trk.stage_ms_mean()
        c = out.counts.cpu().numpy()
        ms = float(sum(st))
        print(f"cfg {cfg}: clusters {ev.n} seeds {int(c[3])} tracks {int(c[0])} | {ms:.3f} ms/call "
              f"{ev.n / ms / 1e6:.3f} G clusters/s | a1..a5 ms {[round(float(x), 3) for x in st]} | "
              f"grid {trk.grid_shape()} | scratch {trk.scratch_bytes() / 1e9:.2f} GB", flush=True)
        trk.close()


if __name__ == "__main__":
    main(sys.argv[1:])
