"""CPU-side checks of the boundary: the C-ABI library loads without a GPU and exports every symbol
include/tpc_track.h declares; host-only entry points behave; the product never touches oracle/;
bench.py's multi-rank bookkeeping works over gloo with world_size 2."""
import ctypes as C
import os
import re
import socket
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2502_09138_b200 import build, load_library
    build.build()
    return load_library()


def test_library_exports_every_declared_symbol(lib):
    from paper_2502_09138_b200 import declared_symbols
    names = declared_symbols()
    assert {"tpc_tracker_create", "tpc_track", "tpc_tracker_destroy", "tpc_track_host"} <= set(names)
    for s in names:
        assert hasattr(lib, s), s


def test_struct_layouts_match_header():
    from paper_2502_09138_b200.binding import Params, TrackRec, TRACK_DTYPE, _Geometry, _TracksOut, _Clusters
    assert C.sizeof(TrackRec) == 112 == TRACK_DTYPE.itemsize
    assert C.sizeof(Params) == 10 * 4 + 12 * 8
    assert C.sizeof(_Clusters) == 24 and C.sizeof(_TracksOut) == 32
    assert C.sizeof(_Geometry) == 8 + 8 + 4 * 8 + 8


def test_default_params_are_the_survey_constants(lib):
    """Appendix A of SURVEY.md; the oracle holds its own copy -- both must state the same written definition."""
    from paper_2502_09138_b200.binding import default_params
    from oracle import oracle
    p, q = default_params(), oracle.default_params()
    assert (p.w_y, p.w_z, p.cost_wy, p.cost_wz, p.c_max, p.l_min) == (1280, 1600, 9, 4, 3538944, 5)
    assert (p.max_miss, p.n_min_tracklet, p.n_min_owned) == (5, 10, 10)
    assert (p.sigma_y, p.sigma_z, p.sinphi_max, p.gate_d, p.gate_y_cm, p.gate_z_cm) == (0.1, 0.15, 0.95, 15.0, 2.0, 2.5)
    assert list(p.c_reset) == [0.25, 0.25, 0.05, 0.05, 25.0] and p.cq_per_tesla == -0.00299792458
    for f in ("w_y", "w_z", "cost_wy", "cost_wz", "c_max", "l_min", "max_miss", "n_min_tracklet", "n_min_owned",
              "sigma_y", "sigma_z", "sinphi_max", "gate_d", "gate_y_cm", "gate_z_cm", "cq_per_tesla"):
        assert getattr(p, f) == getattr(q, f), f
    assert list(p.c_reset) == list(q.c_reset)


def test_host_only_entry_points(lib):
    assert lib.tpc_status_string(0) == b"ok"
    for code in (-1, -2, -3, -4, -5):
        assert lib.tpc_status_string(code) not in (b"ok", b"unknown status")
    assert lib.tpc_status_string(-99) == b"unknown status"
    h = C.c_void_p()
    assert lib.tpc_tracker_create(None, None, C.byref(h)) == -1          # TPC_ERR_ARG, before any CUDA call
    assert lib.tpc_tracker_destroy(None) == -1
    assert lib.tpc_scratch_bytes(None) == 0 and lib.tpc_launches_per_call(None) == 0


def test_geometry_is_validated_before_cuda(lib):
    """Rows that do not ascend and n_rows < 3 are rejected (TPC_ERR_GEOMETRY) without needing a device.  (Rows of
    unequal pitch are accepted since round 2: P48.)"""
    from paper_2502_09138_b200.binding import _Geometry, _Field
    rx = np.array([85.0, 86.0, 85.5, 89.0])
    g = _Geometry(1, 4, rx.ctypes.data_as(C.POINTER(C.c_double)), 640.0, 0.176, 0.0, 250.0, None)
    f = _Field(0.5)
    h = C.c_void_p()
    assert lib.tpc_tracker_create(C.byref(g), C.byref(f), C.byref(h)) == -2
    g2 = _Geometry(1, 2, rx.ctypes.data_as(C.POINTER(C.c_double)), 640.0, 0.176, 0.0, 250.0, None)
    assert lib.tpc_tracker_create(C.byref(g2), C.byref(f), C.byref(h)) == -2


def test_tracker_fails_loudly_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2502_09138_b200 import Tracker, Geometry
    from gen.events import row_x
    with pytest.raises(RuntimeError, match="no CPU path"):
        Tracker(Geometry(n_sectors=1, row_x=row_x()))


def test_product_never_imports_the_oracle():
    """The oracle is test infrastructure: nothing under the package or include/ may name it."""
    pkg = os.path.join(ROOT, "paper_2502_09138_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if not fn.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                continue
            src = open(os.path.join(dirpath, fn)).read()
            assert not re.search(r"^\s*(from|import)\s+oracle", src, flags=re.M), fn
            assert "tpc_oracle" not in src and "libtpc_oracle" not in src, fn
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".cpp", ".h")):
            src = open(os.path.join(ROOT, "oracle", fn)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_2502_09138_b200", src, flags=re.M), fn
            assert not re.search(r"#include\s*[<\"][^>\"]*(tpc_track\.h|tpc_internal)", src), fn
            assert "libtpctrack" not in src, fn


def test_bench_gpus_flag_starts_replica_ranks_gloo_world2():
    """`bench.py --gpus 2` outside torchrun starts two replica ranks itself (torchrun's environment, rendezvous on
    127.0.0.1).  N > 1: ranks are replicas on their own events (weak scaling, no data-path collective); rank 0 reports
    the max-over-ranks time and the sum of units.  Run on the CPU over gloo through the launcher."""
    import json
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_PORT")}
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--selftest-ranks",
                          "--batch-events", "4"], capture_output=True, text=True, timeout=300, env=env)
    assert out.returncode == 0, out.stderr
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line == {"selftest": "ranks", "n_gpus": 2, "ms_max": 15.0, "units_sum": 300.0, "seeds_distinct": True}


def test_bench_under_torchrun_environment_does_not_spawn_again():
    """With torchrun's variables already set, --gpus N is only a label: the process is one rank of the job."""
    import json
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE="2", LOCAL_RANK=str(r), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--selftest-ranks"],
                                      env=env, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True))
    outs = [p.communicate(timeout=240)[0] for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    line = json.loads([l for l in outs[0].splitlines() if l.startswith("{")][-1])
    assert line["n_gpus"] == 2 and line["seeds_distinct"] and line["units_sum"] == 300.0


def test_bench_reference_arm_prints_contract_line():
    import json
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                          "--warmup", "0"], capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "clusters/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
