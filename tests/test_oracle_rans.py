"""Pins for the oracle's entropy stage (NEXT-3, readings P57..P60 in DESIGN.md; "TPC rANS Encoding").

The paper names the coder and nothing else; the pins are what the mathematics fixes: values worked out by hand,
closed forms (a certain symbol costs nothing, a symbol of probability 2^-k costs exactly k bits), the Shannon bound
on the size, and losslessness.
"""
import numpy as np
import pytest

from oracle import oracle as orc

M = 65536


def test_p57_symbol_mapping_worked():
    # A = 16: values -7 .. 7 are the symbols 1 .. 15, everything else is the escape symbol 0
    assert [orc.rans_symbol(v, 4) for v in (-7, -1, 0, 1, 7)] == [1, 7, 8, 9, 15]
    assert [orc.rans_symbol(v, 4) for v in (-8, 8, 100000, -2**31, 2**31 - 1)] == [0, 0, 0, 0, 0]
    # A = 4096: the residual streams
    assert orc.rans_symbol(-2047, 12) == 1 and orc.rans_symbol(2047, 12) == 4095 and orc.rans_symbol(2048, 12) == 0


def test_p58_normalisation_worked():
    # counts (3, 1): K = 2, f = 1 + floor(n * 65534 / 4) = (49151, 16384), sum 65535, the remainder 1 goes to the
    # most frequent symbol
    assert list(orc.rans_normalise([3, 1])) == [49152, 16384]
    # three equal counts and a symbol that does not occur: 1 + floor(65533 / 3) = 21845 each, the remainder 1 goes
    # to the first of the equals; the absent symbol keeps 0
    assert list(orc.rans_normalise([1, 0, 1, 1])) == [21846, 0, 21845, 21845]
    # one symbol: certain
    assert list(orc.rans_normalise([0, 0, 7, 0])) == [0, 0, M, 0]
    # nothing at all
    assert list(orc.rans_normalise([0, 0, 0, 0])) == [0, 0, 0, 0]


def test_p58_normalisation_properties():
    rng = np.random.default_rng(5)
    for trial in range(50):
        A = int(rng.choice([2, 16, 256, 4096]))
        counts = rng.integers(0, 1000, A) * (rng.random(A) < rng.uniform(0.05, 1.0))
        if trial % 7 == 0:
            counts[rng.integers(0, A)] += 10**9          # one dominating symbol
        if trial % 5 == 0:
            counts = np.minimum(counts, 1)               # many symbols that occur once
        counts = counts.astype(np.int64)
        if counts.sum() == 0:
            counts[0] = 1
        f = orc.rans_normalise(counts).astype(np.int64)
        assert f.sum() == M
        assert np.array_equal(f > 0, counts > 0)
        # proportional up to the rounding of the rule: f_s - 1 <= n_s M / N, and only the top symbol gets more
        N, K = counts.sum(), int((counts > 0).sum())
        top = int(np.argmax(counts))
        others = np.arange(A) != top
        assert np.all(f[others] <= 1 + counts[others] * (M - K) // N)
        assert np.all(f[others] >= (counts[others] > 0) * 1)
        assert 0 <= f[top] - (1 + counts[top] * (M - K) // N) < max(K, 1)


def test_p59_worked_chunk_without_emission():
    # A = 4: values 0, 0, 0, 1 are the symbols 2, 2, 2, 3 with f = (49152, 16384), c = (0, 49152) (P58 above).
    # Backwards from x = 65536:
    #   s = 3: x = floor(65536 / 16384) * 65536 + 0 + 49152              = 311296
    #   s = 2: x = floor(311296 / 49152) * 65536 + 311296 mod 49152 + 0  = 6 * 65536 + 16384 = 409600
    #   s = 2: x = floor(409600 / 49152) * 65536 + 16384                 = 8 * 65536 + 16384 = 540672
    #   s = 2: x = floor(540672 / 49152) * 65536 + 0                     = 11 * 65536        = 720896 = 0x000B0000
    enc = orc.rans_encode([0, 0, 0, 1], alphabet_bits=2, chunk=4)
    assert list(enc["freq"]) == [0, 0, 49152, 16384]
    assert list(enc["payload"]) == [0x00, 0x00, 0x0B, 0x00]
    assert list(enc["chunk_off"]) == [0, 4] and list(enc["esc_off"]) == [0, 0]
    assert list(orc.rans_decode(enc)) == [0, 0, 0, 1]


def test_p59_p60_worked_chunk_with_an_emission_and_escapes():
    # A = 4: values -1, 0, 1, 5 twice = symbols 1, 2, 3, 0 (5 escapes) twice; four symbols with two occurrences each:
    # f = 1 + floor(2 * 65532 / 8) = 16384 each, c = (0, 16384, 32768, 49152).  Backwards from 0x10000, every step
    # is x = (x >> 14) << 16 | (x & 16383) + c_s:
    #   s=0: 0x40000, s=3: 0x10C000, s=2: 0x438000, s=1: 0x10E4000, s=0: 0x4390000, s=3: 0x10E4C000, s=2: 0x43938000;
    #   before the last symbol x >= 16384 * 65536: emit 0x8000, x = 0x4393; s=1: 65536 + 915 + 16384 = 0x14393.
    # Layout: the state, little endian, then the word.
    v = [-1, 0, 1, 5, -1, 0, 1, 5]
    enc = orc.rans_encode(v, alphabet_bits=2, chunk=8)
    assert list(enc["freq"]) == [16384] * 4
    assert list(enc["payload"]) == [0x93, 0x43, 0x01, 0x00, 0x00, 0x80]
    assert list(enc["escapes"]) == [5, 5]
    assert list(orc.rans_decode(enc)) == v
    # the same stream in chunks of 3: three chunks, the escapes are attributed to the chunks that hold them
    enc3 = orc.rans_encode(v, alphabet_bits=2, chunk=3)
    assert list(enc3["esc_off"]) == [0, 0, 1, 2]
    assert len(enc3["chunk_off"]) == 4 and enc3["chunk_off"][-1] == len(enc3["payload"])
    assert list(orc.rans_decode(enc3)) == v


def test_a_certain_symbol_costs_nothing():
    # closed form: f = M leaves the state where it is, x = floor(x / M) M + x mod M: four bytes of state per chunk
    enc = orc.rans_encode(np.full(1000, 3, np.int32), alphabet_bits=12, chunk=128)
    assert len(enc["payload"]) == 4 * 8
    assert list(enc["payload"][:4]) == [0x00, 0x00, 0x01, 0x00]
    assert np.array_equal(orc.rans_decode(enc), np.full(1000, 3))


def test_a_symbol_of_probability_one_sixteenth_costs_four_bits():
    # closed form: 16 symbols, equally often: f = 1 + floor(65520 / 16) = 4096 = M / 16 each; a step multiplies the
    # state by 16 exactly (four bits inserted), so starting from 17 bits a word leaves at every fourth symbol:
    # a chunk of 512 symbols is 128 words + the state = 260 bytes, whatever the order of the symbols
    rng = np.random.default_rng(2)
    v = np.tile(np.arange(-8, 8, dtype=np.int32), 512 * 5 // 16)
    rng.shuffle(v)
    enc = orc.rans_encode(v, alphabet_bits=5, chunk=512)
    assert set(enc["freq"][enc["freq"] > 0]) == {4096}
    assert np.array_equal(np.diff(enc["chunk_off"].astype(np.int64)), np.full(5, 260))
    assert np.array_equal(orc.rans_decode(enc), v)


@pytest.mark.parametrize("n,chunk,bits", [(0, 16, 8), (1, 16, 8), (15, 16, 8), (16, 16, 8), (17, 16, 8), (1000, 1, 4),
                                          (5000, 512, 12), (4097, 4096, 12), (20000, 333, 6)])
def test_round_trip_is_lossless(n, chunk, bits):
    rng = np.random.default_rng(n + chunk)
    v = np.rint(rng.normal(0, (1 << bits) / 6.0, n)).astype(np.int32)      # tails beyond the alphabet escape
    if n > 10:
        v[rng.integers(0, n, 5)] = rng.integers(-2**31, 2**31 - 1, 5, dtype=np.int64).astype(np.int32)
    enc = orc.rans_encode(v, alphabet_bits=bits, chunk=chunk)
    n_chunks = (n + chunk - 1) // chunk
    assert len(enc["chunk_off"]) == n_chunks + 1 and enc["chunk_off"][0] == 0
    assert int(enc["chunk_off"][-1]) == len(enc["payload"])
    half = 1 << (bits - 1)
    esc = v[(v <= -half) | (v >= half)]
    assert np.array_equal(enc["escapes"], esc)                               # stream order
    assert int(enc["freq"].astype(np.int64).sum()) == (M if n else 0)
    assert np.array_equal(orc.rans_decode(enc), v)


def test_size_meets_the_shannon_bound_of_the_table():
    # the coded size is the information content under the normalised table, sum log2(M / f_s), plus what a chunk
    # carries on top: 32 bits of state, of which 16 are the initial x = 2^16, and less than one word of slack
    rng = np.random.default_rng(11)
    for sigma, chunk in ((3.0, 512), (60.0, 512), (60.0, 64), (400.0, 2048)):
        v = np.rint(rng.normal(0, sigma, 200000)).astype(np.int32)
        enc = orc.rans_encode(v, alphabet_bits=12, chunk=chunk)
        f = enc["freq"].astype(np.float64)
        sym = np.where((v > -2048) & (v < 2048), v + 2048, 0)
        ideal_bits = float(np.sum(np.log2(M / f[sym])))
        n_chunks = len(enc["chunk_off"]) - 1
        bits = 8.0 * len(enc["payload"])
        assert bits >= ideal_bits + 16 * n_chunks - 1e-6
        assert bits <= ideal_bits * 1.001 + 48 * n_chunks
        # and the table is close to the empirical distribution: within 1 % of the empirical entropy
        cnt = np.bincount(sym, minlength=4096).astype(np.float64)
        p = cnt[cnt > 0] / cnt.sum()
        h_emp = float(-(p * np.log2(p)).sum()) * len(v)
        assert ideal_bits <= h_emp * 1.01 + 64


def test_the_two_boundaries_of_the_rules():
    # P57: -A/2 itself is outside the alphabet (its slot is the escape symbol's): it must travel in the escape list
    v = np.array([-8, 7, -7, 8, -8, 0], np.int32)
    enc = orc.rans_encode(v, alphabet_bits=4, chunk=4)
    assert list(enc["escapes"]) == [-8, 8, -8] and list(enc["esc_off"]) == [0, 2, 3]
    assert np.array_equal(orc.rans_decode(enc), v)
    # P59: x = f 2^16 exactly must emit (x = 2^16 meets a symbol of frequency 1 at the end of a chunk); without the
    # emission the step would leave the state at 2^32 + c_s
    v = np.zeros(70000, np.int32)
    v[-1] = 1
    enc = orc.rans_encode(v, alphabet_bits=4, chunk=70000)
    assert enc["freq"][8] == M - 1 and enc["freq"][9] == 1
    # by hand: emit 0x0000, x = 1; x = 1 * 65536 + 0 + c_9 = 65536 + 65535 = 0x1FFFF; the 69999 symbols of
    # frequency M - 1 then shrink nothing below 2^16 and add < 1 word in total: no further emission
    assert np.array_equal(orc.rans_decode(enc), v)
    assert len(enc["payload"]) in (6, 8)
    assert list(enc["payload"][-2:]) == [0x00, 0x00]          # the word emitted first is consumed last
