"""ctypes binding of include/tpc_track.h.  Same names as the C ABI; torch supplies device memory and streams.

No arithmetic of the method lives here.  Nothing here imports oracle/.
"""
from __future__ import annotations

import ctypes as C
import os
import re
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_HEADER = os.path.join(os.path.dirname(_HERE), "include", "tpc_track.h")


def lib_path() -> str:
    return os.path.join(_HERE, "libtpctrack.so")


class Params(C.Structure):
    """tpc_params_t"""
    _fields_ = [
        ("w_y", C.c_int32), ("w_z", C.c_int32), ("cost_wy", C.c_int32), ("cost_wz", C.c_int32),
        ("c_max", C.c_int32), ("l_min", C.c_int32), ("max_miss", C.c_int32), ("n_min_tracklet", C.c_int32),
        ("n_min_owned", C.c_int32), ("reserved", C.c_int32),
        ("sigma_y", C.c_double), ("sigma_z", C.c_double), ("sinphi_max", C.c_double), ("gate_d", C.c_double),
        ("gate_y_cm", C.c_double), ("gate_z_cm", C.c_double), ("c_reset", C.c_double * 5),
        ("cq_per_tesla", C.c_double),
    ]


class _Geometry(C.Structure):
    _fields_ = [
        ("n_sectors", C.c_int32), ("n_rows", C.c_int32), ("row_x", C.POINTER(C.c_double)),
        ("units_per_cm", C.c_double), ("y_half_tan", C.c_double), ("y_half_cm", C.c_double),
        ("z_extent_cm", C.c_double), ("params", C.POINTER(Params)),
    ]


class _Field(C.Structure):
    _fields_ = [("bz_tesla", C.c_double)]


class _Clusters(C.Structure):
    _fields_ = [("y", C.c_void_p), ("z", C.c_void_p), ("row_offsets", C.c_void_p)]


class TrackRec(C.Structure):
    """tpc_track_rec_t (112 bytes)"""
    _fields_ = [
        ("x", C.c_float), ("y", C.c_float), ("z", C.c_float), ("sinphi", C.c_float), ("tanl", C.c_float),
        ("qpt", C.c_float), ("cov", C.c_float * 15), ("chi2", C.c_float), ("sector", C.c_int32),
        ("first_row", C.c_int32), ("last_row", C.c_int32), ("n_hits", C.c_int32), ("hit_offset", C.c_int32),
        ("seed_cluster", C.c_int32),
    ]


TRACK_DTYPE = np.dtype([
    ("x", "<f4"), ("y", "<f4"), ("z", "<f4"), ("sinphi", "<f4"), ("tanl", "<f4"), ("qpt", "<f4"),
    ("cov", "<f4", (15,)), ("chi2", "<f4"), ("sector", "<i4"), ("first_row", "<i4"), ("last_row", "<i4"),
    ("n_hits", "<i4"), ("hit_offset", "<i4"), ("seed_cluster", "<i4"),
])
assert TRACK_DTYPE.itemsize == C.sizeof(TrackRec) == 112


class MergeParams(C.Structure):
    """tpc_merge_params_t"""
    _fields_ = [("gap_max", C.c_int32), ("n_per_side", C.c_int32), ("chi2_max", C.c_double),
                ("sector_angle", C.c_double)]


class _Compressed(C.Structure):
    """tpc_compressed_t"""
    _fields_ = [("drow", C.c_void_p), ("ry", C.c_void_p), ("rz", C.c_void_p), ("hist_ry", C.c_void_p),
                ("hist_rz", C.c_void_p), ("hist_drow", C.c_void_p)]


class _RansStream(C.Structure):
    """tpc_rans_stream_t"""
    _fields_ = [("freq", C.c_void_p), ("chunk_off", C.c_void_p), ("esc_off", C.c_void_p), ("payload", C.c_void_p),
                ("escapes", C.c_void_p), ("counts", C.c_void_p), ("payload_capacity", C.c_int64),
                ("escape_capacity", C.c_int64)]


class ClusterParams(C.Structure):
    """tpc_cluster_params_t"""
    _fields_ = [("n_pads", C.c_int32), ("n_per_side", C.c_int32), ("pad_units", C.c_int32), ("time_units", C.c_int32),
                ("q_peak_min", C.c_int32)]


class _Digits(C.Structure):
    _fields_ = [("pad", C.c_void_p), ("time", C.c_void_p), ("adc", C.c_void_p), ("offsets", C.c_void_p)]


class _ClustersOut(C.Structure):
    _fields_ = [("y", C.c_void_p), ("z", C.c_void_p), ("qtot", C.c_void_p), ("qmax", C.c_void_p),
                ("row_offsets", C.c_void_p), ("counts", C.c_void_p), ("capacity", C.c_int32)]


class _TracksOut(C.Structure):
    _fields_ = [("tracks", C.c_void_p), ("track_capacity", C.c_int32), ("hit_capacity", C.c_int32),
                ("hit_ids", C.c_void_p), ("counts", C.c_void_p)]


def declared_symbols() -> list[str]:
    """Every function include/tpc_track.h declares (used by the ABI test)."""
    src = open(_HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(tpc_[a-z_0-9]+)\s*\(", src)))


_lib = None


def load_library():
    """Loads libtpctrack.so.  Raises if it has not been built: there is no fallback path."""
    global _lib
    if _lib is not None:
        return _lib
    p = lib_path()
    if not os.path.exists(p):
        raise RuntimeError(f"{p} is missing: build it with `python -m paper_2502_09138_b200.build` "
                           "(the CUDA library is the only implementation; there is no CPU fallback)")
    lib = C.CDLL(p)
    lib.tpc_default_params.argtypes = [C.POINTER(Params)]
    lib.tpc_default_params.restype = None
    lib.tpc_tracker_create.argtypes = [C.POINTER(_Geometry), C.POINTER(_Field), C.POINTER(C.c_void_p)]
    lib.tpc_track.argtypes = [C.c_void_p, C.POINTER(_Clusters), C.c_int64, C.c_void_p, C.POINTER(_TracksOut)]
    lib.tpc_track_host.argtypes = lib.tpc_track.argtypes
    lib.tpc_refit.argtypes = [C.c_void_p, C.POINTER(_Clusters), C.c_int64, C.c_void_p, C.POINTER(_TracksOut),
                              C.c_void_p]
    lib.tpc_default_merge_params.argtypes = [C.POINTER(MergeParams)]
    lib.tpc_default_merge_params.restype = None
    lib.tpc_merge.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.POINTER(MergeParams), C.c_void_p,
                              C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.tpc_refit_merged.argtypes = [C.c_void_p, C.POINTER(_Clusters), C.c_int64, C.c_void_p, C.POINTER(_TracksOut),
                                     C.c_void_p, C.c_void_p, C.POINTER(MergeParams), C.c_void_p]
    lib.tpc_compress.argtypes = [C.c_void_p, C.POINTER(_Clusters), C.c_int64, C.c_void_p, C.POINTER(_TracksOut),
                                 C.POINTER(_Compressed)]
    lib.tpc_decompress.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(_TracksOut), C.POINTER(_Compressed), C.c_void_p,
                                   C.c_void_p, C.c_void_p]
    lib.tpc_rans_encode.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_int64, C.c_int32, C.c_int32, C.c_void_p,
                                    C.POINTER(_RansStream)]
    lib.tpc_rans_decode.argtypes = [C.c_void_p, C.POINTER(_RansStream), C.c_int64, C.c_int32, C.c_int32, C.c_void_p,
                                    C.c_void_p, C.c_int32]
    lib.tpc_rans_encode_static.argtypes = [C.c_void_p, C.c_int32, C.c_int64, C.c_int32, C.c_int32, C.c_void_p,
                                           C.POINTER(_RansStream)]
    lib.tpc_default_cluster_params.argtypes = [C.POINTER(ClusterParams)]
    lib.tpc_default_cluster_params.restype = None
    lib.tpc_clusterize.argtypes = [C.c_void_p, C.POINTER(_Digits), C.c_int64, C.POINTER(ClusterParams), C.c_void_p,
                                   C.POINTER(_ClustersOut)]
    lib.tpc_tracker_destroy.argtypes = [C.c_void_p]
    lib.tpc_status_string.argtypes = [C.c_int]
    lib.tpc_status_string.restype = C.c_char_p
    lib.tpc_last_cuda_error.argtypes = [C.c_void_p]
    lib.tpc_last_cuda_error.restype = C.c_char_p
    lib.tpc_scratch_bytes.argtypes = [C.c_void_p]
    lib.tpc_scratch_bytes.restype = C.c_int64
    lib.tpc_launches_per_call.argtypes = [C.c_void_p]
    lib.tpc_reserve_seeds.argtypes = [C.c_void_p, C.c_int64]
    lib.tpc_set_concurrency.argtypes = [C.c_void_p, C.c_int32]
    lib.tpc_debug_set_a4_variant.argtypes = [C.c_void_p, C.c_int]
    lib.tpc_debug_set_a2_variant.argtypes = [C.c_void_p, C.c_int]
    lib.tpc_set_stage_timing.argtypes = [C.c_void_p, C.c_int]
    lib.tpc_get_stage_ms.argtypes = [C.c_void_p, C.POINTER(C.c_float)]
    lib.tpc_get_stage_ms_mean.argtypes = [C.c_void_p, C.POINTER(C.c_float), C.POINTER(C.c_int32)]
    lib.tpc_debug_copy_links.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.tpc_debug_copy_seeds.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.tpc_debug_copy_tracklets.argtypes = [C.c_void_p] + [C.c_void_p] * 6
    lib.tpc_debug_copy_owner.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
    lib.tpc_debug_grid_info.argtypes = [C.c_void_p] + [C.POINTER(C.c_int32)] * 4
    lib.tpc_debug_copy_grid.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    _lib = lib
    return lib


def default_params() -> Params:
    p = Params()
    load_library().tpc_default_params(C.byref(p))
    return p


class TpcError(RuntimeError):
    def __init__(self, status: int, detail: str = ""):
        self.status = status
        msg = load_library().tpc_status_string(status).decode()
        super().__init__(f"tpc status {status}: {msg}" + (f" ({detail})" if detail else ""))


@dataclass
class Geometry:
    """tpc_geometry_t as Python values."""
    n_sectors: int
    row_x: np.ndarray
    units_per_cm: float = 640.0
    y_half_tan: float = float(np.tan(np.deg2rad(10.0)))
    y_half_cm: float = 0.0
    z_extent_cm: float = 250.0
    params: Params | None = None
    bz_tesla: float = 0.5


@dataclass
class TracksOut:
    """Device buffers written by tpc_track (torch tensors) plus helpers to read them on the host."""
    tracks: "object"      # torch.uint8 [track_capacity * 112]
    hit_ids: "object"     # torch.int32 [hit_capacity]
    counts: "object"      # torch.int32 [4]

    def to_host(self):
        import torch
        torch.cuda.synchronize(self.counts.device)
        c = self.counts.cpu().numpy()
        nt, nh, flags, ns = int(c[0]), int(c[1]), int(c[2]), int(c[3])
        if flags:
            raise RuntimeError(f"output overflow flags={flags}: tracks={nt} hits={nh}")
        trk = self.tracks[: nt * 112].cpu().numpy().view(TRACK_DTYPE)
        hits = self.hit_ids[:nh].cpu().numpy()
        return trk, hits, ns


def _ptr(t) -> int:
    return 0 if t is None else int(t.data_ptr())


class Tracker:
    """tpc_tracker_create / tpc_track / tpc_tracker_destroy."""

    def __init__(self, geo: Geometry):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2502_09138_b200 needs a CUDA device (sm_100a); there is no CPU path")
        self._lib = load_library()
        torch.cuda.init()
        torch.zeros(1, device="cuda")   # make sure the primary context exists before the library touches it
        self.geo = geo
        rx = np.ascontiguousarray(geo.row_x, dtype=np.float64)
        g = _Geometry(int(geo.n_sectors), int(rx.shape[0]), rx.ctypes.data_as(C.POINTER(C.c_double)),
                      float(geo.units_per_cm), float(geo.y_half_tan), float(geo.y_half_cm), float(geo.z_extent_cm),
                      C.pointer(geo.params) if geo.params is not None else None)
        f = _Field(float(geo.bz_tesla))
        h = C.c_void_p()
        rc = self._lib.tpc_tracker_create(C.byref(g), C.byref(f), C.byref(h))
        if rc != 0:
            raise TpcError(rc)
        self._h = h
        self.n_rows = int(rx.shape[0])
        self.n_sectors = int(geo.n_sectors)
        self.l_min = int(geo.params.l_min) if geo.params is not None else 5

    def close(self):
        if getattr(self, "_h", None):
            self._lib.tpc_tracker_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc):
        if rc != 0:
            raise TpcError(rc, self._lib.tpc_last_cuda_error(self._h).decode())

    @staticmethod
    def _stream_ptr(stream):
        import torch
        s = stream if stream is not None else torch.cuda.current_stream()
        return C.c_void_p(int(s.cuda_stream))

    def alloc_out(self, n: int, track_capacity: int | None = None, hit_capacity: int | None = None) -> TracksOut:
        import torch
        tc = int(track_capacity if track_capacity is not None else n // 10 + 16)
        hc = int(hit_capacity if hit_capacity is not None else n + 16)
        return TracksOut(torch.empty(tc * 112, dtype=torch.uint8, device="cuda"),
                         torch.empty(hc, dtype=torch.int32, device="cuda"),
                         torch.zeros(4, dtype=torch.int32, device="cuda"))

    def track(self, y, z, row_offsets, out: TracksOut | None = None, stream=None) -> TracksOut:
        """tpc_track: y, z int32 CUDA tensors [n]; row_offsets int32/uint32-valued CUDA tensor
        [n_sectors*n_rows + 1] (torch has no uint32 arithmetic; the bits are what the library reads).
        Asynchronous on `stream` (default: torch's current stream)."""
        import torch
        assert y.is_cuda and z.is_cuda and row_offsets.is_cuda
        assert y.dtype == torch.int32 and z.dtype == torch.int32 and row_offsets.dtype in (torch.int32, torch.uint32)
        assert y.is_contiguous() and z.is_contiguous() and row_offsets.is_contiguous()
        n = int(y.shape[0])
        assert int(z.shape[0]) == n and int(row_offsets.shape[0]) == self.n_sectors * self.n_rows + 1
        if out is None:
            out = self.alloc_out(n)
        cl = _Clusters(_ptr(y), _ptr(z), _ptr(row_offsets))
        o = _TracksOut(_ptr(out.tracks), int(out.tracks.shape[0] // 112), int(out.hit_ids.shape[0]),
                       _ptr(out.hit_ids), _ptr(out.counts))
        self._check(self._lib.tpc_track(self._h, C.byref(cl), C.c_int64(n), self._stream_ptr(stream), C.byref(o)))
        return out

    def refit(self, y, z, row_offsets, out: "TracksOut", stream=None):
        """tpc_refit on the output of the last track() call with the same inputs; returns a device uint8 tensor of
        track records (same layout as out.tracks)."""
        import torch
        n = int(y.shape[0])
        cl = _Clusters(_ptr(y), _ptr(z), _ptr(row_offsets))
        o = _TracksOut(_ptr(out.tracks), int(out.tracks.shape[0] // 112), int(out.hit_ids.shape[0]), _ptr(out.hit_ids),
                       _ptr(out.counts))
        ref = torch.zeros_like(out.tracks)
        self._check(self._lib.tpc_refit(self._h, C.byref(cl), C.c_int64(n), self._stream_ptr(stream), C.byref(o),
                                        _ptr(ref)))
        return ref

    def merge(self, tracks, counts, params: "MergeParams | None" = None, stream=None):
        """tpc_merge on device track records (uint8 tensor of 112-byte records, e.g. out.tracks or the tensor refit()
        returned) and the int32[4] counts of that call.  Returns device tensors (succ, pred, link_chi2, merge_counts)."""
        import torch
        cap = int(tracks.shape[0] // 112)
        succ = torch.empty(max(cap, 1), dtype=torch.int32, device=tracks.device)
        pred = torch.empty(max(cap, 1), dtype=torch.int32, device=tracks.device)
        chi2 = torch.empty(max(cap, 1), dtype=torch.float32, device=tracks.device)
        mc = torch.zeros(4, dtype=torch.int32, device=tracks.device)
        self._check(self._lib.tpc_merge(self._h, _ptr(tracks), _ptr(counts), C.c_int32(cap),
                                        C.byref(params) if params is not None else None, self._stream_ptr(stream),
                                        _ptr(succ), _ptr(pred), _ptr(chi2), _ptr(mc)))
        return succ, pred, chi2, mc

    def refit_merged(self, y, z, row_offsets, out: "TracksOut", succ, pred, params: "MergeParams | None" = None,
                     stream=None):
        """tpc_refit_merged: refit over every chain of linked tracks (succ / pred from merge()); returns a device uint8
        tensor of track records (heads carry the result, other tracks n_hits = 0)."""
        import torch
        n = int(y.shape[0])
        cl = _Clusters(_ptr(y), _ptr(z), _ptr(row_offsets))
        o = _TracksOut(_ptr(out.tracks), int(out.tracks.shape[0] // 112), int(out.hit_ids.shape[0]), _ptr(out.hit_ids),
                       _ptr(out.counts))
        ref = torch.zeros_like(out.tracks)
        self._check(self._lib.tpc_refit_merged(self._h, C.byref(cl), C.c_int64(n), self._stream_ptr(stream), C.byref(o),
                                               _ptr(succ), _ptr(pred),
                                               C.byref(params) if params is not None else None, _ptr(ref)))
        return ref

    def compress(self, y, z, row_offsets, out: "TracksOut", stream=None):
        """tpc_compress on the output of the last track() call: dict of device tensors drow (uint8), ry, rz (int32) in
        hit-list order and the histograms hist_ry, hist_rz (65536), hist_drow (256)."""
        import torch
        dev = out.hit_ids.device
        hc = int(out.hit_ids.shape[0])
        c = dict(drow=torch.zeros(max(hc, 1), dtype=torch.uint8, device=dev),
                 ry=torch.zeros(max(hc, 1), dtype=torch.int32, device=dev),
                 rz=torch.zeros(max(hc, 1), dtype=torch.int32, device=dev),
                 hist_ry=torch.zeros(65536, dtype=torch.int32, device=dev),
                 hist_rz=torch.zeros(65536, dtype=torch.int32, device=dev),
                 hist_drow=torch.zeros(256, dtype=torch.int32, device=dev))
        cl = _Clusters(_ptr(y), _ptr(z), _ptr(row_offsets))
        o = _TracksOut(_ptr(out.tracks), int(out.tracks.shape[0] // 112), hc, _ptr(out.hit_ids), _ptr(out.counts))
        cs = _Compressed(*[_ptr(c[k]) for k in ("drow", "ry", "rz", "hist_ry", "hist_rz", "hist_drow")])
        self._check(self._lib.tpc_compress(self._h, C.byref(cl), C.c_int64(int(y.shape[0])), self._stream_ptr(stream),
                                           C.byref(o), C.byref(cs)))
        return c

    def decompress(self, out: "TracksOut", comp: dict, stream=None):
        """tpc_decompress: (row, y, z) int32 device tensors in hit-list order from the residual streams."""
        import torch
        dev = out.hit_ids.device
        hc = int(out.hit_ids.shape[0])
        row, yy, zz = (torch.zeros(max(hc, 1), dtype=torch.int32, device=dev) for _ in range(3))
        o = _TracksOut(_ptr(out.tracks), int(out.tracks.shape[0] // 112), hc, _ptr(out.hit_ids), _ptr(out.counts))
        cs = _Compressed(*[_ptr(comp[k]) for k in ("drow", "ry", "rz", "hist_ry", "hist_rz", "hist_drow")])
        self._check(self._lib.tpc_decompress(self._h, self._stream_ptr(stream), C.byref(o), C.byref(cs), _ptr(row),
                                             _ptr(yy), _ptr(zz)))
        return row, yy, zz

    @staticmethod
    def _rans_struct(enc: dict) -> "_RansStream":
        return _RansStream(_ptr(enc["freq"]), _ptr(enc["chunk_off"]), _ptr(enc["esc_off"]), _ptr(enc["payload"]),
                           _ptr(enc["escapes"]), _ptr(enc["counts"]), int(enc["payload"].shape[0]),
                           int(enc["escapes"].shape[0]))

    def rans_encode(self, values, alphabet_bits: int = 12, chunk: int = 512, payload_capacity=None,
                    escape_capacity=None, stream=None, into: "dict | None" = None):
        """tpc_rans_encode of an int32 or uint8 CUDA tensor: dict of device tensors freq, chunk_off, esc_off (uint32
        bits in int32), payload (uint8), escapes (int32), counts (int64[4]: payload bytes, escapes, chunks, flags).
        Default capacities hold any input; `into` reuses the buffers of an earlier call of the same shape."""
        import torch
        n = int(values.shape[0])
        vb = {torch.int32: 4, torch.uint8: 1}[values.dtype]
        n_chunks = (n + chunk - 1) // chunk
        dev = values.device
        enc = into
        if enc is None:
            pc = int(payload_capacity if payload_capacity is not None else 4 * n_chunks + 2 * n)
            ec = int(escape_capacity if escape_capacity is not None else n)
            enc = dict(freq=torch.zeros(1 << alphabet_bits, dtype=torch.int32, device=dev),
                       chunk_off=torch.zeros(n_chunks + 1, dtype=torch.int32, device=dev),
                       esc_off=torch.zeros(n_chunks + 1, dtype=torch.int32, device=dev),
                       payload=torch.zeros(max(pc, 2), dtype=torch.uint8, device=dev),
                       escapes=torch.zeros(max(ec, 1), dtype=torch.int32, device=dev),
                       counts=torch.zeros(4, dtype=torch.int64, device=dev),
                       n=n, alphabet_bits=alphabet_bits, chunk=chunk, value_bytes=vb)
            if payload_capacity is not None:
                enc["payload"] = enc["payload"][:pc] if pc >= 2 else enc["payload"][:0]
            if escape_capacity is not None:
                enc["escapes"] = enc["escapes"][:ec]
        rs = self._rans_struct(enc)
        self._check(self._lib.tpc_rans_encode(self._h, C.c_void_p(_ptr(values)), vb, C.c_int64(n), alphabet_bits, chunk,
                                              self._stream_ptr(stream), C.byref(rs)))
        return enc

    def rans_decode(self, enc: dict, stream=None):
        """tpc_rans_decode: the values of an encoded stream (same dtype as the input of rans_encode)."""
        import torch
        n = enc["n"]
        vb = enc["value_bytes"]
        values = torch.zeros(max(n, 1), dtype=torch.int32 if vb == 4 else torch.uint8, device=enc["freq"].device)
        rs = self._rans_struct(enc)
        self._check(self._lib.tpc_rans_decode(self._h, C.byref(rs), C.c_int64(n), enc["alphabet_bits"], enc["chunk"],
                                              self._stream_ptr(stream), C.c_void_p(_ptr(values)), vb))
        return values[:n]

    def clusterize(self, pad, time, adc, offsets, n_pads: int, params: "ClusterParams | None" = None, capacity=None,
                   stream=None):
        """tpc_clusterize: digits (uint16 CUDA tensors pad, time, adc; int32 CSR offsets) -> dict of device tensors
        y, z, qtot, qmax (int32), row_offsets (int32 bits of uint32), counts (int32[2])."""
        import torch
        nd = int(pad.shape[0])
        cap = int(capacity if capacity is not None else max(nd // 3, 16))
        dev = offsets.device
        out = dict(y=torch.zeros(cap, dtype=torch.int32, device=dev), z=torch.zeros(cap, dtype=torch.int32, device=dev),
                   qtot=torch.zeros(cap, dtype=torch.int32, device=dev), qmax=torch.zeros(cap, dtype=torch.int32, device=dev),
                   row_offsets=torch.zeros(self.n_sectors * self.n_rows + 1, dtype=torch.int32, device=dev),
                   counts=torch.zeros(2, dtype=torch.int32, device=dev))
        if params is None:
            params = ClusterParams()
            self._lib.tpc_default_cluster_params(C.byref(params))
        params.n_pads = int(n_pads)
        d = _Digits(_ptr(pad), _ptr(time), _ptr(adc), _ptr(offsets))
        o = _ClustersOut(_ptr(out["y"]), _ptr(out["z"]), _ptr(out["qtot"]), _ptr(out["qmax"]), _ptr(out["row_offsets"]),
                         _ptr(out["counts"]), cap)
        self._check(self._lib.tpc_clusterize(self._h, C.byref(d), C.c_int64(nd), C.byref(params),
                                             self._stream_ptr(stream), C.byref(o)))
        return out

    def track_host(self, y, z, row_offsets, tracks, hit_ids, counts, stream=None):
        """tpc_track_host: all arguments are HOST tensors (pinned for asynchronous copies): y, z int32 [n],
        row_offsets int32 [R+1], tracks uint8 [cap*112], hit_ids int32 [cap], counts int32 [4].
        Returns after the results are in the host buffers."""
        n = int(y.shape[0])
        assert not y.is_cuda and not tracks.is_cuda
        cl = _Clusters(_ptr(y), _ptr(z), _ptr(row_offsets))
        o = _TracksOut(_ptr(tracks), int(tracks.shape[0] // 112), int(hit_ids.shape[0]), _ptr(hit_ids), _ptr(counts))
        self._check(self._lib.tpc_track_host(self._h, C.byref(cl), C.c_int64(n), self._stream_ptr(stream), C.byref(o)))

    # ---- bookkeeping ----
    def scratch_bytes(self) -> int:
        return int(self._lib.tpc_scratch_bytes(self._h))

    def launches_per_call(self) -> int:
        return int(self._lib.tpc_launches_per_call(self._h))

    def set_stage_timing(self, enable: bool):
        self._check(self._lib.tpc_set_stage_timing(self._h, 1 if enable else 0))

    def stage_ms(self):
        ms = (C.c_float * 5)()
        self._check(self._lib.tpc_get_stage_ms(self._h, ms))
        return [float(v) for v in ms]

    def stage_ms_mean(self):
        """(mean ms per stage a1..a5, number of calls averaged) since set_stage_timing(True)."""
        ms = (C.c_float * 5)()
        n = C.c_int32()
        self._check(self._lib.tpc_get_stage_ms_mean(self._h, ms, C.byref(n)))
        return [float(v) for v in ms], int(n.value)

    # ---- test-only exports (tpc_debug_*) ----
    def debug_links(self, n: int, cleaned: bool):
        import torch
        up = torch.empty(n, dtype=torch.int32, device="cuda")
        dn = torch.empty(n, dtype=torch.int32, device="cuda")
        self._check(self._lib.tpc_debug_copy_links(self._h, 1 if cleaned else 0, _ptr(up), _ptr(dn), self._stream_ptr(None)))
        return up.cpu().numpy(), dn.cpu().numpy()

    def set_concurrency(self, k: int):
        """tpc_set_concurrency: how many tpc_track calls the caller keeps in flight on the device at the same time."""
        self._check(self._lib.tpc_set_concurrency(self._h, int(k)))

    def reserve_seeds(self, n_seeds: int):
        """tpc_reserve_seeds: raise the handle's seed capacity (after TPC_FLAG_SEED_OVERFLOW)."""
        self._check(self._lib.tpc_reserve_seeds(self._h, C.c_int64(int(n_seeds))))

    def set_a4_variant(self, variant: int):
        """tpc_debug_set_a4_variant: 0 = by call size, 1 = uniform kernel, 2 = phase kernels (tests)."""
        self._check(self._lib.tpc_debug_set_a4_variant(self._h, C.c_int(int(variant))))

    def set_a2_variant(self, variant: int):
        """tpc_debug_set_a2_variant: 0 = direct, 1 = rows staged in shared memory by TMA bulk copies."""
        self._check(self._lib.tpc_debug_set_a2_variant(self._h, C.c_int(int(variant))))

    def debug_seeds(self, n: int, n_seeds: int):
        import torch
        cap = max(int(n_seeds), 1)
        st = torch.empty(cap, dtype=torch.int32, device="cuda")
        ln = torch.empty(cap, dtype=torch.int32, device="cuda")
        self._check(self._lib.tpc_debug_copy_seeds(self._h, _ptr(st), _ptr(ln), self._stream_ptr(None)))
        return st[:n_seeds].cpu().numpy(), ln[:n_seeds].cpu().numpy()

    def debug_tracklets(self, n_seeds: int):
        import torch
        ns = max(n_seeds, 1)
        par = torch.empty(ns * 6, dtype=torch.float32, device="cuda")
        cov = torch.empty(ns * 15, dtype=torch.float32, device="cuda")
        chi2 = torch.empty(ns, dtype=torch.float32, device="cuda")
        nh = torch.empty(ns, dtype=torch.int32, device="cuda")
        hits = torch.empty(ns * self.n_rows, dtype=torch.int32, device="cuda")
        self._check(self._lib.tpc_debug_copy_tracklets(self._h, _ptr(par), _ptr(cov), _ptr(chi2), _ptr(nh), _ptr(hits),
                                                       self._stream_ptr(None)))
        return (par.cpu().numpy().reshape(ns, 6)[:n_seeds], cov.cpu().numpy().reshape(ns, 15)[:n_seeds],
                chi2.cpu().numpy()[:n_seeds], nh.cpu().numpy()[:n_seeds],
                hits.cpu().numpy().reshape(ns, self.n_rows)[:n_seeds])

    def debug_owner(self, n: int):
        import torch
        o = torch.empty(n, dtype=torch.int32, device="cuda")
        self._check(self._lib.tpc_debug_copy_owner(self._h, _ptr(o), self._stream_ptr(None)))
        return o.cpu().numpy()

    def grid_shape(self):
        """Grid of the most recent call (api.cu: choose_grid): bins-per-row stride, nz, shift_y, shift_z."""
        vals = [C.c_int32() for _ in range(4)]
        self._check(self._lib.tpc_debug_grid_info(self._h, *[C.byref(v) for v in vals]))
        stride, nz, sy, sz = [int(v.value) for v in vals]
        return dict(stride=stride, nz=nz, shift_y=sy, shift_z=sz)

    def debug_grid(self, n: int):
        import torch
        vals = [C.c_int32() for _ in range(4)]
        self._check(self._lib.tpc_debug_grid_info(self._h, *[C.byref(v) for v in vals]))
        stride, nz, sy, sz = [int(v.value) for v in vals]
        ids = torch.empty(n, dtype=torch.int32, device="cuda")
        bs = torch.empty(self.n_sectors * self.n_rows * stride, dtype=torch.int32, device="cuda")
        self._check(self._lib.tpc_debug_copy_grid(self._h, _ptr(ids), _ptr(bs), self._stream_ptr(None)))
        return dict(stride=stride, nz=nz, shift_y=sy, shift_z=sz, ids=ids.cpu().numpy(),
                    bin_start=bs.cpu().numpy().view(np.uint32).reshape(self.n_sectors * self.n_rows, stride))


RANS_STATIC_SCRATCH_BYTES = 4 << 20     # TPC_RANS_STATIC_SCRATCH_BYTES


def rans_encode_static(values, enc: dict, stream=None) -> dict:
    """tpc_rans_encode_static: the encoder that allocates nothing (its scratch is a fixed array inside the library, at
    most RANS_STATIC_SCRATCH_BYTES per call; all calls share it, so calls must not overlap on the GPU).  `enc` holds
    the caller's output tensors, laid out as Tracker.rans_encode returns them (freq, chunk_off, esc_off, payload,
    escapes, counts and n, alphabet_bits, chunk, value_bytes); it is written and returned.  Needs no Tracker."""
    import torch
    n = int(values.shape[0])
    vb = {torch.int32: 4, torch.uint8: 1}[values.dtype]
    if n != enc["n"] or vb != enc["value_bytes"]:
        raise ValueError("enc was laid out for another input")
    rs = Tracker._rans_struct(enc)
    s = stream if stream is not None else torch.cuda.current_stream()
    rc = load_library().tpc_rans_encode_static(C.c_void_p(_ptr(values)), vb, C.c_int64(n), enc["alphabet_bits"],
                                               enc["chunk"], C.c_void_p(int(s.cuda_stream)), C.byref(rs))
    if rc != 0:
        raise TpcError(rc)
    return enc


def rans_alloc(n: int, alphabet_bits: int = 12, chunk: int = 512, value_bytes: int = 4, device="cuda") -> dict:
    """Output tensors of an encode call for n values, sized so that any input fits (what Tracker.rans_encode makes)."""
    import torch
    n_chunks = (n + chunk - 1) // chunk
    return dict(freq=torch.zeros(1 << alphabet_bits, dtype=torch.int32, device=device),
                chunk_off=torch.zeros(n_chunks + 1, dtype=torch.int32, device=device),
                esc_off=torch.zeros(n_chunks + 1, dtype=torch.int32, device=device),
                payload=torch.zeros(max(4 * n_chunks + 2 * n, 2), dtype=torch.uint8, device=device),
                escapes=torch.zeros(max(n, 1), dtype=torch.int32, device=device),
                counts=torch.zeros(4, dtype=torch.int64, device=device),
                n=n, alphabet_bits=alphabet_bits, chunk=chunk, value_bytes=value_bytes)

