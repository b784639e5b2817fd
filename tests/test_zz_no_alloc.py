"""tpc_rans_encode_static: the one entry point that allocates nothing (scratch = a fixed array inside the library).

Collected last on purpose (the suite runs with pytest -x).  Checks the new entry point against the existing
tpc_rans_encode path -- integer work, so byte for byte -- on calls in a row that share the static array: a large
input first, then a smaller one of another alphabet and chunk size (stale slots, histogram and counts of the first call
must not leak into the second), then the first again.  Self-contained: no fixture, passes alone in a fresh process.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _same(a, b, label):
    import torch
    ca, cb = a["counts"].cpu().numpy(), b["counts"].cpu().numpy()
    assert ca.tolist() == cb.tolist() and int(ca[3]) == 0, (label, ca, cb)
    nb, ne = int(ca[0]), int(ca[1])
    for key in ("freq", "chunk_off", "esc_off"):
        assert torch.equal(a[key], b[key]), (label, key)
    assert torch.equal(a["payload"][:nb], b["payload"][:nb]), label
    assert torch.equal(a["escapes"][:ne], b["escapes"][:ne]), label


def test_static_scratch_encoder_equals_the_allocating_path_on_calls_in_a_row():
    import torch
    from gen.events import row_x
    from paper_2502_09138_b200 import Tracker, rans_alloc, rans_encode_static, RANS_STATIC_SCRATCH_BYTES
    from paper_2502_09138_b200.binding import Geometry, TpcError
    rng = np.random.default_rng(17)
    trk = Tracker(Geometry(n_sectors=1, row_x=row_x()))          # only the existing path needs a handle
    cases = []
    for n, bits, chunk, dtype in ((1_500_000, 12, 512, np.int32), (70_001, 6, 333, np.int32), (200_000, 8, 100, np.uint8),
                                  (1, 12, 512, np.int32), (1_500_000, 12, 512, np.int32)):
        if dtype == np.uint8:
            v = rng.integers(0, 256, n).astype(np.uint8)
        else:
            v = np.rint(rng.normal(0, (1 << bits) / 6.0, n)).astype(np.int32)     # tails escape
            if n > 10:
                v[rng.integers(0, n, 5)] = rng.integers(-2**31, 2**31 - 1, 5, dtype=np.int64).astype(np.int32)
        cases.append((torch.from_numpy(v).cuda(), bits, chunk))
    for k, (d, bits, chunk) in enumerate(cases):
        ref = trk.rans_encode(d, alphabet_bits=bits, chunk=chunk)
        enc = rans_alloc(int(d.shape[0]), bits, chunk, value_bytes=d.element_size())
        enc["payload"].fill_(0xEE)
        rans_encode_static(d, enc)
        _same(enc, ref, (k, int(d.shape[0]), bits, chunk))
        assert torch.equal(trk.rans_decode(enc), d), k              # and it decodes to the input
    # the same buffers again, twice back to back without a synchronisation in between (one stream: serialised)
    d, bits, chunk = cases[0]
    ref = trk.rans_encode(d, alphabet_bits=bits, chunk=chunk)
    e1 = rans_alloc(int(d.shape[0]), bits, chunk)
    e2 = rans_alloc(int(d.shape[0]), bits, chunk)
    rans_encode_static(d, e1)
    rans_encode_static(d, e2)
    _same(e1, ref, "back to back 1")
    _same(e2, ref, "back to back 2")
    # beyond the static array: a clear error, nothing enqueued
    n_big = RANS_STATIC_SCRATCH_BYTES // 2 + 4096
    big = torch.zeros(n_big, dtype=torch.int32, device="cuda")
    enc = rans_alloc(n_big, 12, 512)
    enc["counts"].fill_(-5)
    with pytest.raises(TpcError) as ei:
        rans_encode_static(big, enc)
    assert ei.value.status == -6 and "static" in str(ei.value)
    torch.cuda.synchronize()
    assert enc["counts"].cpu().tolist() == [-5, -5, -5, -5]
    trk.close()
