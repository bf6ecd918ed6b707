"""Pins for the entropy-stage oracle (oracle/tmd_ans_oracle.c, oracle/tmd_ans.py) against things other than itself.

PAPER.md L20 names the coder ("lossless ANS"), L49 / L68 place it just before track-model decoding; it prints no stream, so
the pins are: streams derived BY HAND from the published coding function (Duda, arXiv:1311.2540:
x' = floor(x/f) 2^12 + c + x mod f, 16-bit renormalisation), the Shannon bound on the compressed size, a second,
independent model of the whole block coder in Python integers (written from DESIGN.md §10, shares nothing with oracle/),
and decode(encode(x)) == x on skewed, uniform and degenerate planes and on whole containers.
"""
import math

import numpy as np
import pytest

from oracle import tmd_ans as A
from oracle import tmd_oracle as O
from tmd_inputs import physical as ph
from tmd_inputs.adversarial import random_compressed
from tmd_inputs.layout import COMPRESSED_FIELDS

L, M, LANES = 1 << 16, 1 << 12, 32


def table(**f):
    t = np.zeros(256, np.uint16)
    for k, v in f.items():
        t[int(k[1:])] = v
    assert int(t.sum()) == M
    return t


def split(block: np.ndarray):
    return block[:128].view(np.uint32).tolist(), block[128:].view(np.uint16).tolist()


# ------------------------------------------------------------------------------------------------ hand-derived streams
def test_one_symbol_alphabet_emits_nothing():
    # f = 4096, c = 0:  x' = floor(x/4096) 4096 + x mod 4096 = x.  No state ever changes, none reaches 2^20 f = 2^32, so
    # the block is the 32 initial states 2^16 and not a single word -- whatever the number of symbols.
    for n in (1, 31, 32, 33, 1000, 8192):
        blk = A.encode_block(np.full(n, 7, np.uint8), table(s7=4096))
        assert len(blk) == 128 and split(blk)[0] == [L] * 32
        assert A.decode_block(blk, n, table(s7=4096)).tolist() == [7] * n


def test_three_symbols_one_per_coder():
    # symbols 0 (f 2048, c 0), 1 (f 1024, c 2048), 2 (f 1024, c 3072) in coders 0, 1, 2, each starting from x = 2^16 < 2^20 f:
    #   coder 0: floor(65536/2048) 4096 + 0    + 0 = 32 * 4096        = 131072
    #   coder 1: floor(65536/1024) 4096 + 2048 + 0 = 64 * 4096 + 2048 = 264192
    #   coder 2: floor(65536/1024) 4096 + 3072 + 0 = 64 * 4096 + 3072 = 265216
    t = table(s0=2048, s1=1024, s2=1024)
    states, words = split(A.encode_block(np.array([0, 1, 2], np.uint8), t))
    assert states == [131072, 264192, 265216] + [L] * 29 and words == []
    assert A.decode_block(A.encode_block(np.array([0, 1, 2], np.uint8), t), 3, t).tolist() == [0, 1, 2]


def test_renormalisation_word_by_hand():
    # D = symbol 9 (f 1, c 4095), A = symbol 4 (f 4095, c 0).  33 symbols: D at k = 0 and k = 32 (both coder 0), A elsewhere.
    # The encoder runs backwards.  Coder 0: k = 32 first: x = 65536 < 2^20 * 1 -> no word; x' = 65536 * 4096 + 4095 =
    # 268439551 (0x10000FFF).  Then k = 0: x >= 2^20 -> emit the low word 0x0FFF = 4095, x = 0x1000 = 4096;
    # x' = 4096 * 4096 + 4095 = 16781311.  Coders 1..31 (one A each): floor(65536/4095) = 16, 65536 mod 4095 = 16 ->
    # x' = 16 * 4096 + 0 + 16 = 65552.  One word in the stream.
    t = table(s9=1, s4=4095)
    sym = np.full(33, 4, np.uint8); sym[0] = sym[32] = 9
    blk = A.encode_block(sym, t)
    states, words = split(blk)
    assert states == [16781311] + [65552] * 31 and words[:1] == [4095] and len(blk) == 128 + 4
    got, trace = A.decode_block(blk, 33, t, want_trace=True)
    assert got.tolist() == sym.tolist()
    # decoder, coder 0: slot 4095 -> D, x = 1 * 4096 + 4095 - 4095 = 4096 < 2^16 -> x = 4096 * 65536 + 4095; then D again -> 2^16
    assert int(trace[0]) == 268439551 and int(trace[32]) == L and all(int(v) == L for v in trace[1:32])


# ------------------------------------------------------------------------------------------------ independent integer model
def model_encode(sym, freq):
    """The block coder restated with Python integers from DESIGN.md §10 (no numpy, no oracle): returns (states, words)."""
    cum = [0] * 257
    for s in range(256):
        cum[s + 1] = cum[s] + int(freq[s])
    x = [L] * LANES
    emitted = []
    for k in range(len(sym) - 1, -1, -1):
        lane, s = k % LANES, int(sym[k])
        f, c = int(freq[s]), cum[s]
        if x[lane] >= (1 << 20) * f:
            emitted.append(x[lane] & 0xFFFF)
            x[lane] >>= 16
        x[lane] = (x[lane] // f) * M + c + x[lane] % f
    return x, emitted[::-1]


@pytest.mark.parametrize("seed,n,p", [(1, 8192, 0.25), (2, 5000, 0.02), (3, 97, 0.5), (4, 1, 0.3), (5, 8192, 0.9)])
def test_block_coder_equals_the_integer_model(seed, n, p):
    rng = np.random.default_rng(seed)
    sym = np.minimum(rng.geometric(p, n) - 1, 255).astype(np.uint8)
    freq = A.build_table(sym)
    assert int(freq.sum()) == M and np.all(freq[np.unique(sym)] >= 1)
    blk = A.encode_block(sym, freq)
    states, words = split(blk)
    want_states, want_words = model_encode(sym, freq)
    assert states == want_states and words[:len(want_words)] == want_words and len(words) - len(want_words) in (0, 1)
    assert np.array_equal(A.decode_block(blk, n, freq), sym)


# ------------------------------------------------------------------------------------------------ Shannon bound
@pytest.mark.parametrize("p", [0.05, 0.3, 0.8])
def test_compressed_size_meets_the_entropy_of_the_quantised_table(p):
    rng = np.random.default_rng(11)
    n = 200_000
    sym = np.minimum(rng.geometric(p, n) - 1, 255).astype(np.uint8)
    freq = A.build_table(sym)
    cnt = np.bincount(sym, minlength=256)
    bits = -sum(int(c) * math.log2(int(f) / M) for c, f in zip(cnt, freq) if c)        # n * cross-entropy of the stored table
    n_blocks = (n + A.BLOCK - 1) // A.BLOCK
    payload = sum(len(A.encode_block(sym[i:i + A.BLOCK], freq)) for i in range(0, n, A.BLOCK))
    # every coder carries its final state (32 bits, of which >= 16 are information of the stream) -> at most 128 B per block
    assert bits / 8 - 4 * n_blocks <= payload <= bits / 8 + 132 * n_blocks
    ideal = -sum(int(c) * math.log2(c / n) for c in cnt if c)
    assert bits <= ideal * 1.01 + 64                                               # 12-bit quantisation costs < 1 %


# ------------------------------------------------------------------------------------------------ round trips
@pytest.mark.parametrize("kind", ["uniform", "constant", "two_values", "all_256", "empty"])
def test_plane_round_trip(kind):
    rng = np.random.default_rng(3)
    sym = {"uniform": rng.integers(0, 256, 30_000), "constant": np.full(9000, 200), "two_values": rng.integers(0, 2, 20_001) * 255,
           "all_256": np.concatenate((np.arange(256), np.zeros(50_000, int))), "empty": np.zeros(0, int)}[kind].astype(np.uint8)
    freq = A.build_table(sym)
    for i in range(0, len(sym), A.BLOCK):
        blk = A.encode_block(sym[i:i + A.BLOCK], freq)
        assert np.array_equal(A.decode_block(blk, len(sym[i:i + A.BLOCK]), freq), sym[i:i + A.BLOCK])


def test_container_round_trip_and_compression(geo2, geo36):
    ev = ph.generate_event(ph.config0(), geo2)
    comp = O.encode(geo2, 0.5, ev.trk_ncl, ev.trk_qptf, ev.att, ev.leg, ev.un)
    blob = A.encode_container(comp)
    back = A.decode_container(blob)
    for k in COMPRESSED_FIELDS:
        assert np.array_equal(getattr(back, k), getattr(comp, k)), k
    assert blob.size < 0.8 * comp.nbytes()                    # track-model residuals are small numbers: they compress
    rnd = random_compressed(geo36, 300, 4000, 5)
    back = A.decode_container(A.encode_container(rnd))
    for k in COMPRESSED_FIELDS:
        assert np.array_equal(getattr(back, k), getattr(rnd, k)), k


def test_truncated_block_is_reported():
    rng = np.random.default_rng(8)
    sym = rng.integers(0, 256, 4000).astype(np.uint8)
    freq = A.build_table(sym)
    blk = A.encode_block(sym, freq)
    with pytest.raises(RuntimeError):
        A.decode_block(blk[: len(blk) // 2], 4000, freq)


# ------------------------------------------------------------------------------------------------ the library's host encoder
def test_library_host_encoder_writes_containers_the_oracle_decodes(geo2, geo36):
    # two independent encoders (oracle/tmd_ans.py and the library's tmd_entropy_encode_host, which share no code) must both
    # write valid TMDZ: the oracle decoder restores the input from the library's container.  Runs without a GPU.
    from paper_2411_02206_b200 import tmd as T
    ev = ph.generate_event(ph.config0(), geo2)
    for comp, n_bins in ((O.encode(geo2, 0.5, ev.trk_ncl, ev.trk_qptf, ev.att, ev.leg, ev.un), geo2.n_bins),
                         (random_compressed(geo36, 200, 3000, 6), geo36.n_bins),
                         (random_compressed(geo36, 0, 0, 7), geo36.n_bins)):
        arrays = {k: np.ascontiguousarray(getattr(comp, k)) for k in COMPRESSED_FIELDS}
        blob = T.tmd_entropy_encode_host(arrays, n_bins)
        assert T.tmd_entropy_sizes(blob[:64])[:4] == (comp.n_tracks, comp.n_attached, comp.n_unattached, n_bins)
        back = A.decode_container(blob)
        for k in COMPRESSED_FIELDS:
            assert np.array_equal(getattr(back, k), getattr(comp, k)), k
        assert len(blob) <= T.tmd_entropy_bound(comp.n_tracks, comp.n_attached, comp.n_unattached, n_bins)
        # the two encoders agree on the size within the freedom of the table quantisation
        assert abs(len(blob) - len(A.encode_container(comp))) <= 0.01 * len(blob) + 64
