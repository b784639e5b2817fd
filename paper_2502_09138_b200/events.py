"""Glue between a synthetic event (gen.events.Event, duck-typed) and the binding: geometry + device upload.
Holds no arithmetic of the method."""
from __future__ import annotations

import numpy as np

from .binding import Geometry, Params


def geometry_from_event(ev, params: Params | None = None) -> Geometry:
    open_sector = bool(getattr(ev.cfg, "open_sector", False))
    return Geometry(
        n_sectors=int(ev.n_sectors), row_x=np.asarray(ev.row_x, dtype=np.float64), units_per_cm=640.0,
        y_half_tan=float(np.tan(np.deg2rad(10.0))), y_half_cm=160.0 if open_sector else 0.0,
        z_extent_cm=float(ev.z_extent_cm) + 2.0, params=params, bz_tesla=float(ev.cfg.bz))


def upload(ev, device="cuda"):
    """(y, z, row_offsets) as CUDA tensors; row_offsets keeps its uint32 bits in an int32 tensor."""
    import torch
    y = torch.from_numpy(np.ascontiguousarray(ev.y, dtype=np.int32)).to(device)
    z = torch.from_numpy(np.ascontiguousarray(ev.z, dtype=np.int32)).to(device)
    ro = torch.from_numpy(np.ascontiguousarray(ev.row_offsets, dtype=np.uint32).view(np.int32)).to(device)
    return y, z, ro
