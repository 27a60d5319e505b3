"""Pins of the oracle against things other than itself (SURVEY.md §8(c) "What pins it"):
paper-printed widths, closed-form sizes, hand-typed bytes, brute-force b (independent
Python builder), second-witness decoder, round trips and walk-the-headers invariants.
CPU only."""
import itertools
import os
import struct

import numpy as np
import pytest

from oracle import witness

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    with open(os.path.join(GOLD, name)) as f:
        return [ln.split() for ln in f if ln.strip() and not ln.startswith("#")]


def _dt(W):
    return np.uint32 if W == 32 else np.uint64


# ---------------------------------------------------------------- width helper
def test_paper_widths(oracle_mod):
    for mx, mn, w in _rows("paper_widths.txt"):
        assert oracle_mod.width(int(mx) - int(mn)) == int(w)


def test_width_closed_forms(oracle_mod):
    assert oracle_mod.width(0) == 0
    for k in range(1, 64):
        assert oracle_mod.width((1 << k) - 1) == k
        assert oracle_mod.width(1 << k) == k + 1
    assert oracle_mod.width((1 << 64) - 1) == 64


# ---------------------------------------------------------------- sizes
def test_closed_form_sizes(oracle_mod):
    for W, n, gap, total in _rows("closed_form_sizes.txt"):
        W, n, gap, total = int(W), int(n), int(gap), int(total)
        x = (1000 + gap * np.arange(n, dtype=np.uint64)).astype(_dt(W))
        s = oracle_mod.compress(x)
        assert len(s) == total, (W, n, gap)
        assert len(s) <= oracle_mod.compress_bound(n, W)
        assert np.array_equal(oracle_mod.decompress(s, W), x)


def test_block_bytes_formula(oracle_mod):
    # typed independently from FORMAT.md
    assert oracle_mod.block_bytes(0, 0, 32) == 16
    assert oracle_mod.block_bytes(1, 1, 32) == 16 + 16 + 16      # pos 1->4, high 4 => 8 -> 16
    assert oracle_mod.block_bytes(1, 3, 32) == 16 + 16 + 16      # 4 + 12 = 16
    assert oracle_mod.block_bytes(1, 4, 32) == 16 + 16 + 32      # 4 + 16 = 20 -> 32
    assert oracle_mod.block_bytes(5, 7, 64) == 16 + 80 + 64      # 8 + 56 = 64
    assert oracle_mod.block_bytes(64, 0, 64) == 16 + 1024
    for W in (32, 64):
        for b in range(W + 1):
            for n in range(128):
                assert oracle_mod.block_bytes(b, n, W) == witness.block_bytes(b, n, W)


def test_compress_bound_is_worst_case(oracle_mod):
    rng = np.random.default_rng(0)
    for W in (32, 64):
        x = rng.integers(0, 1 << W, size=1000, dtype=np.uint64).astype(_dt(W))   # incompressible
        s = oracle_mod.compress(x)
        assert len(s) <= oracle_mod.compress_bound(1000, W)
        assert np.array_equal(oracle_mod.decompress(s, W), x)


# ---------------------------------------------------------------- bytes
def test_hand_vector(oracle_mod):
    want = bytes.fromhex(_rows("hand_vector_2000_2127.hex")[0][0])
    got = oracle_mod.compress(np.arange(2000, 2128, dtype=np.uint32)).tobytes()
    assert got == want


def test_exception_block_by_hand(oracle_mod):
    # gap-1 block with one step of 2^20 at j=77: b=1, n_exc=1, block = 16+16+16 = 48 B
    gaps = np.ones(128, dtype=np.uint64)
    gaps[77] = 1 << 20
    x = (np.cumsum(gaps) + 5).astype(np.uint32)
    s = oracle_mod.compress(x).tobytes()
    assert len(s) == 32 + 16 + 48
    blk = s[48:]
    assert blk[8] == 1 and blk[9] == 1
    # bit 77//4=19 of column 77%4=1 is the LOW bit of 2^20, i.e. 0
    words = struct.unpack("<4I", blk[16:32])
    assert words == (0xFFFFFFFE, 0xFFFFFFFF & ~(1 << 19), 0xFFFFFFFF, 0xFFFFFFFF)
    assert blk[32] == 77 and blk[33:36] == bytes(3)
    assert struct.unpack("<I", blk[36:40])[0] == (1 << 20) >> 1
    assert blk[40:48] == bytes(8)
    assert np.array_equal(oracle_mod.decompress(np.frombuffer(s, np.uint8), 32), x)


def test_paper_sequence8(oracle_mod):
    seq = [int(t) for t in _rows("paper_seq8.txt")[0]]
    x = np.array(seq, dtype=np.uint64)
    s = oracle_mod.compress(x)
    assert np.array_equal(oracle_mod.decompress(s, 64), x)
    assert witness.decode_stream(s.tobytes(), 64) == seq
    # the 8th value does not fit 32 bits: as u32 it is reduced mod 2^32 and still round-trips
    x32 = x.astype(np.uint32)
    assert np.array_equal(oracle_mod.decompress(oracle_mod.compress(x32), 32), x32)
    # tiny block degenerates to an exception list: b = 0, 7 exceptions (d_0 = 0 is none)
    blk = s.tobytes()[48:]
    assert blk[8] == 0 and blk[9] == 7 and len(blk) == 16 + 64


# ---------------------------------------------------------------- choice of b
def _check_b(oracle_mod, d, W):
    d = [int(v) for v in d]
    b, n_exc = oracle_mod.choose_b(np.array(d, dtype=np.uint64), W)
    bb, size = witness.brute_force_b(d, W)
    assert (b, oracle_mod.block_bytes(b, n_exc, W)) == (bb, size), d[:8]
    assert oracle_mod.emit_block(np.array(d, dtype=np.uint64), 12345, b, W) == witness.build_block(d, 12345, b, W)


def test_choose_b_exhaustive_small_alphabets(oracle_mod):
    # all blocks whose first L deltas come from a small alphabet (rest 0), both widths
    for alphabet, L in (((0, 1, 1 << 9), 5), ((1, 3, 1 << 31), 4), ((2, 1 << 40, (1 << 64) - 1), 3)):
        for W in (32, 64):
            if W == 32 and max(alphabet) >= 1 << 32:
                continue
            for combo in itertools.product(alphabet, repeat=L):
                d = [0] + list(combo) + [0] * (127 - L)
                _check_b(oracle_mod, d, W)


def test_choose_b_random(oracle_mod):
    rng = np.random.default_rng(1)
    for trial in range(60):
        W = 32 if trial % 2 else 64
        bits = int(rng.integers(1, W + 1))
        d = rng.integers(0, 1 << min(bits, 62), size=128, dtype=np.uint64)
        k = int(rng.integers(0, 12))                       # sprinkle outliers
        for p in rng.integers(1, 128, size=k):
            d[p] = int(rng.integers(0, 1 << 62)) >> int(rng.integers(0, 62 - min(W, 62) + 1) + (62 - min(W, 62)))
        d[0] = 0
        if W == 32:
            d &= np.uint64(0xFFFFFFFF)
        _check_b(oracle_mod, d, W)


def test_forced_b_blocks_decode(oracle_mod):
    # any b in 0..W is decodable, not only the canonical one
    rng = np.random.default_rng(2)
    for W in (32, 64):
        d = rng.integers(0, 1 << 20, size=128, dtype=np.uint64)
        d[0] = 0
        d[100] = (1 << (W - 1)) + 3
        want = ((np.cumsum(d.astype(object)) + 7) % (1 << W))
        for b in (0, 1, 7, 20, 21, 32, W):
            blk = oracle_mod.emit_block(d, 7, b, W)
            assert blk == witness.build_block([int(v) for v in d], 7, b, W)
            hdr = b"BFSC" + bytes([1, W, 1, 0]) + struct.pack("<QQI", 128, 48 + len(blk), 1) + bytes(4)
            s = hdr + struct.pack("<II", 3, 3 + len(blk) // 16) + bytes(8) + blk
            got = oracle_mod.decompress(np.frombuffer(s, np.uint8), W)
            assert [int(v) for v in got] == [int(v) for v in want]
            assert witness.decode_stream(s, W) == [int(v) for v in want]
