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


# ---------------------------------------------------------------- mode 2: BP128-D1 (FORMAT.md §7)
def _bp128_case(name, W, n):
    dt = _dt(W)
    if name == "gap1":
        return (1000 + np.arange(n, dtype=np.uint64)).astype(dt)
    if name == "gap3":
        return (1000 + 3 * np.arange(n, dtype=np.uint64)).astype(dt)
    if name == "step20":
        x = 7 + np.arange(n, dtype=np.uint64)
        x[51:] += (1 << 20) - 1                        # delta of ID 51 = 2^20
        return x.astype(dt)
    if name == "seq8":
        return np.array([int(v) for v in _rows("paper_seq8.txt")[0]], dtype=dt)
    if name == "range7":
        return np.arange(2000, 2128, dtype=dt)
    raise KeyError(name)


def test_bp128_sizes_and_witness(oracle_mod):
    for name, W, n, total in _rows("bp128_sizes.txt"):
        W, n, total = int(W), int(n), int(total)
        x = _bp128_case(name, W, n)
        s = oracle_mod.compress(x, codec=oracle_mod.CODEC_BP128)
        assert len(s) == total, name
        assert witness.stream_mode(s.tobytes()) == 2
        assert all(ne == 0 for _, ne in witness.stream_blocks(s.tobytes()))
        assert witness.decode_stream(s.tobytes(), W) == [int(v) for v in x]          # second witness
        assert np.array_equal(oracle_mod.decompress(s, W), x)
        assert len(s) <= oracle_mod.compress_bound(n, W)


def test_bp128_b_is_max_width_and_blocks_match_forced_b(oracle_mod):
    """b = bit length of the widest delta (eq. 6, min = 0), found here with Python's int.bit_length;
    the stream = header(mode 2) | directory | witness.build_block(d, base, b) for every block."""
    rng = np.random.default_rng(11)
    for W in (32, 64):
        for trial in range(12):
            n = int(rng.integers(1, 700))
            hi = int(rng.integers(1, W))
            gaps = rng.integers(0, 1 << int(rng.integers(1, hi + 1)), size=n, dtype=np.uint64)
            gaps[rng.random(n) < 0.03] = rng.integers(0, 1 << hi, dtype=np.uint64)   # outliers: would be exceptions in PFOR
            x = np.cumsum(gaps, dtype=np.uint64).astype(_dt(W))
            s = oracle_mod.compress(x, codec=oracle_mod.CODEC_BP128).tobytes()
            nb = -(-n // 128)
            blocks = witness.stream_blocks(s)
            at = 32 + -(-4 * (nb + 1) // 16) * 16
            for k in range(nb):
                xs = [int(v) for v in x[128 * k:128 * (k + 1)]]
                base, d = witness.deltas_of_block(xs, W)
                b = max(v.bit_length() for v in d)
                assert blocks[k] == (b, 0)
                assert oracle_mod.choose_b_bp128(np.array(d, dtype=np.uint64)) == b
                img = witness.build_block(d, base, b, W)
                assert s[at:at + len(img)] == img
                assert int.from_bytes(s[32 + 4 * k:36 + 4 * k], "little") == at // 16
                at += len(img)
            assert at == len(s) and int.from_bytes(s[16:24], "little") == at
            assert witness.decode_stream(s, W) == [int(v) for v in x]


def test_bp128_equals_pfor_when_no_exception_pays(oracle_mod):
    """Where the PFOR argmin keeps b = maxw in every block the two modes differ in byte 6 only;
    BP128 is never smaller than PFOR (PFOR minimises over a set that contains b = maxw)."""
    x = (5 + 3 * np.arange(5000, dtype=np.uint64)).astype(np.uint32)
    a, b = oracle_mod.compress(x), oracle_mod.compress(x, codec=oracle_mod.CODEC_BP128)
    assert len(a) == len(b) and a[6] == 1 and b[6] == 2
    assert np.array_equal(np.delete(a, 6), np.delete(b, 6))
    rng = np.random.default_rng(5)
    for W in (32, 64):
        g = rng.geometric(1 / 200, size=3000).astype(np.uint64)
        g[rng.random(3000) < 0.01] = 1 << 22
        y = np.cumsum(g, dtype=np.uint64).astype(_dt(W))
        p, q = oracle_mod.compress(y), oracle_mod.compress(y, codec=oracle_mod.CODEC_BP128)
        assert len(p) < len(q)
        assert np.array_equal(oracle_mod.decompress(q, W), y)


def test_bp128_threshold_batch_and_roundtrip(oracle_mod):
    rng = np.random.default_rng(3)
    for W in (32, 64):
        counts = np.array([0, 1, 127, 128, 129, 300, 1000, 5], dtype=np.uint64)
        off = np.concatenate([[0], np.cumsum(counts)]).astype(np.uint64)
        ids = np.cumsum(rng.integers(1, 50, size=int(off[-1]), dtype=np.uint64)).astype(_dt(W))
        for thr in (0, 1024):
            out, out_off = oracle_mod.compress_batch(ids, off, thr, codec=oracle_mod.CODEC_BP128)
            for i, c in enumerate(counts):
                s = out[int(out_off[i]):int(out_off[i + 1])]
                raw = int(c) * W // 8 < thr
                assert s[6] == (0 if raw else 2)                 # RAW selection is independent of the codec
                one = oracle_mod.compress(ids[int(off[i]):int(off[i + 1])], thr, codec=oracle_mod.CODEC_BP128)
                assert np.array_equal(s, one)
            back, id_off = oracle_mod.decompress_batch(out, out_off, W, len(ids))
            assert np.array_equal(back, ids) and np.array_equal(id_off, off)


def test_compress_bound_closed_form(oracle_mod):
    """FORMAT.md §3, pinned from BOTH sides: bound(n, W) == 32 + align16(4 (nb + 1)) + nb (16 + 16 W), typed out
    here, and attained exactly by an incompressible buffer of full blocks (every delta needs W bits)."""
    hand = {(0, 32): 48, (1, 32): 32 + 16 + 528, (128, 32): 32 + 16 + 528, (129, 32): 32 + 16 + 2 * 528,
            (1000, 32): 32 + 48 + 8 * 528, (16384, 32): 32 + 528 + 128 * 528, (1 << 24, 64): 32 + 524304 + 131072 * 1040,
            (0, 64): 48, (127, 64): 32 + 16 + 1040, (385, 64): 32 + 32 + 4 * 1040, (1 << 20, 64): 32 + 32784 + 8192 * 1040,
            (3 * 128, 32): 32 + 16 + 3 * 528}
    for (n, W), want in hand.items():
        nb = -(-n // 128)
        assert want == 32 + -(-4 * (nb + 1) // 16) * 16 + nb * (16 + 16 * W)
        assert oracle_mod.compress_bound(n, W) == want, (n, W)
    for W in (32, 64):                                             # tight: constant gap 2^(W-1) + 1 (mod 2^W) -> every delta is W bits wide
        n = 128 * 5
        x = np.array([(j * ((1 << (W - 1)) + 1)) % (1 << W) for j in range(n)], dtype=np.uint32 if W == 32 else np.uint64)
        s = oracle_mod.compress(x)
        # the first delta of each block is 0, the other 127 have W bits: b = W, no exceptions
        assert len(s) == oracle_mod.compress_bound(n, W)


# ---------------------------------------------------------------- FORMAT.md §8: RAW fallback
def test_raw_fallback_rule(oracle_mod):
    """FORMAT.md §8: with the fallback flag a stream is never larger than its RAW form; it is
    the rule's stream, byte for byte, when that is smaller, and the RAW stream otherwise (ties: RAW). Sizes typed out."""
    F = oracle_mod.FLAG_RAW_FALLBACK
    for W in (32, 64):
        E = W // 8
        dt = _dt(W)
        assert len(oracle_mod.compress(np.zeros(0, dtype=dt), 0, codec=oracle_mod.CODEC_PFOR | F)) == 32          # 48 without
        assert len(oracle_mod.compress(np.array([7], dtype=dt), 0, codec=oracle_mod.CODEC_PFOR | F)) == 32 + 16   # 64 without
        x = (2000 + np.arange(128)).astype(dt)                      # the paper's eq. (7) range: 80 bytes either way
        a, b = oracle_mod.compress(x, 0), oracle_mod.compress(x, 0, codec=oracle_mod.CODEC_PFOR | F)
        assert len(a) == 80 and np.array_equal(a, b)
        inc = np.array([(j * ((1 << (W - 1)) + 1)) % (1 << W) for j in range(640)], dtype=dt)   # every delta W bits wide
        s = oracle_mod.compress(inc, 0, codec=oracle_mod.CODEC_PFOR | F)
        assert len(s) == 32 + 640 * E and s[6] == 0 and s[24:28].view(np.uint32)[0] == 0
        assert np.array_equal(s[32:].view(dt), inc)
        assert len(oracle_mod.compress(inc, 0)) == oracle_mod.compress_bound(640, W) > len(s)
        assert np.array_equal(oracle_mod.decompress(s, W), inc)
        assert witness.decode_stream(s.tobytes(), W) == [int(v) for v in inc]
    # a tie: 128 u32 IDs with a constant gap of 2^29 (30 bits): 32 + 16 + (16 + 16 * 30) = 544 = 32 + 512 -> RAW
    tie = ((np.arange(128, dtype=np.uint64) << np.uint64(29)) & np.uint64(0xFFFFFFFF)).astype(np.uint32)
    assert len(oracle_mod.compress(tie, 0)) == 544
    s = oracle_mod.compress(tie, 0, codec=oracle_mod.CODEC_PFOR | F)
    assert len(s) == 544 and s[6] == 0
    rng = np.random.default_rng(99)
    for _ in range(40):
        W = int(rng.choice([32, 64]))
        n = int(rng.integers(0, 700))
        bits = int(rng.integers(1, W + 1))
        g = rng.integers(0, 1 << min(bits, 63), size=n, dtype=np.uint64)
        x = (np.cumsum(g) & np.uint64((1 << W) - 1)).astype(_dt(W))
        for rule in (oracle_mod.CODEC_PFOR, oracle_mod.CODEC_BP128):
            plain, fb = oracle_mod.compress(x, 0, codec=rule), oracle_mod.compress(x, 0, codec=rule | F)
            raw_total = 32 + -(-n * (W // 8) // 16) * 16
            assert len(fb) == min(len(plain), raw_total) and len(fb) <= raw_total
            assert (fb[6] == 0) == (len(plain) >= raw_total)
            if len(plain) < raw_total:
                assert np.array_equal(fb, plain)
            assert np.array_equal(oracle_mod.decompress(fb, W), x)


# ---------------------------------------------------------------- FORMAT.md §9: frontier bitmaps
def test_bitmap_hand_vector(oracle_mod):
    """The paper's eq. (7) range 2000..2127 as a bitmap, words typed by hand (bit v = bit v % 32 of word v / 32):
    its stream is the hand-typed 80-byte vector of tests/golden/hand_vector_2000_2127.hex; the same bits at
    0..127 with id_base = 2000 give the same bytes."""
    gold = bytes.fromhex("".join(ln.split("#")[0] for ln in open(os.path.join(GOLD, "hand_vector_2000_2127.hex"))).replace(" ", "").replace("\n", ""))
    words = np.zeros(67, dtype=np.uint32)
    words[62] = 0xFFFF0000                                          # bits 2000..2015
    words[63] = words[64] = words[65] = 0xFFFFFFFF                  # bits 2016..2111
    words[66] = 0x0000FFFF                                          # bits 2112..2127
    s = oracle_mod.compress_bitmap(words, 67 * 32, 32)
    assert s.tobytes() == gold
    assert oracle_mod.compress_bitmap(np.full(4, 0xFFFFFFFF, dtype=np.uint32), 128, 32, id_base=2000).tobytes() == gold
    back = np.zeros(67, dtype=np.uint32)
    assert oracle_mod.decompress_to_bitmap(s, 32, back, 67 * 32) == 128 and np.array_equal(back, words)


def test_bitmap_matches_id_list_and_round_trips(oracle_mod):
    """compress_bitmap(bits) == compress(IDs of the set bits), the IDs derived here by numpy (unpackbits, nonzero),
    not by the oracle; n in the header = popcount; decompress_to_bitmap ORs (old bits stay); an ID outside the
    bitmap is DST_TOO_SMALL and leaves the bitmap alone."""
    rng = np.random.default_rng(7)
    for W in (32, 64):
        for n_bits, density in ((1, 1.0), (31, 0.5), (32, 0.5), (1000, 0.5), (4096, 0.02), (70000, 0.3), (5000, 0.0)):
            for id_base in (0, 12345):
                bits = rng.random(n_bits) < density
                words = np.packbits(np.concatenate([bits, np.zeros(-n_bits % 32, dtype=bool)]), bitorder="little").view(np.uint32).copy()
                ids = (np.nonzero(bits)[0].astype(np.uint64) + np.uint64(id_base)).astype(_dt(W))
                s = oracle_mod.compress_bitmap(words, n_bits, W, id_base=id_base)
                assert np.array_equal(s, oracle_mod.compress(ids, 0))
                assert int(s[8:16].view(np.uint64)[0]) == int(bits.sum())
                old = rng.integers(0, 1 << 32, size=len(words), dtype=np.uint64).astype(np.uint32)
                old[-1] &= np.uint32((1 << ((n_bits - 1) % 32 + 1)) - 1)
                back = old.copy()
                assert oracle_mod.decompress_to_bitmap(s, W, back, n_bits, id_base=id_base) == len(ids)
                assert np.array_equal(back, old | words)
                if len(ids) and n_bits > 1:
                    small = old.copy()
                    with pytest.raises(oracle_mod.OracleError) as ei:
                        oracle_mod.decompress_to_bitmap(s, W, small, int(ids[-1]) - id_base, id_base=id_base)   # last ID does not fit
                    assert ei.value.code == oracle_mod.ERR_DST_TOO_SMALL and np.array_equal(small, old)


def test_frontier_update_hand_example_and_set_algebra(oracle_mod):
    """FORMAT.md §9, last item (Algorithm 4 lines 10-13). Hand example: IDs {3, 5, 5, 40}, visited =
    {5, 6}, frontier = {0}: line 11 keeps {3, 40}, line 12 gives visited {3, 5, 6, 40}, line 13 frontier {0, 3, 40}.
    Then the set identities on random inputs, with numpy sets: frontier' = frontier | (S & ~visited),
    visited' = visited | S; the visited bits of other IDs and an out-of-range ID leave everything alone."""
    s = oracle_mod.compress(np.array([3, 5, 5, 40], dtype=np.uint32), 0)
    vis = np.array([(1 << 5) | (1 << 6), 0], dtype=np.uint32)
    fr = np.array([1, 0], dtype=np.uint32)
    assert oracle_mod.decompress_to_frontier(s, 32, fr, vis, 64) == 4
    assert fr.tolist() == [1 | (1 << 3), 1 << 8] and vis.tolist() == [(1 << 3) | (1 << 5) | (1 << 6), 1 << 8]
    rng = np.random.default_rng(11)
    for W in (32, 64):
        for n_bits, dens, id_base in ((1, 1.0, 0), (33, 0.5, 7), (5000, 0.3, 12345), (70000, 0.05, 0)):
            bits = rng.random(n_bits) < dens
            ids = (np.nonzero(bits)[0].astype(np.uint64) + np.uint64(id_base)).astype(_dt(W))
            S = np.packbits(np.concatenate([bits, np.zeros(-n_bits % 32, dtype=bool)]), bitorder="little").view(np.uint32).copy()
            s = oracle_mod.compress(ids, 0)
            tail = np.uint32((1 << ((n_bits - 1) % 32 + 1)) - 1)
            vis0 = rng.integers(0, 1 << 32, size=len(S), dtype=np.uint64).astype(np.uint32); vis0[-1] &= tail
            fr0 = rng.integers(0, 1 << 32, size=len(S), dtype=np.uint64).astype(np.uint32); fr0[-1] &= tail
            vis, fr = vis0.copy(), fr0.copy()
            assert oracle_mod.decompress_to_frontier(s, W, fr, vis, n_bits, id_base=id_base) == len(ids)
            assert np.array_equal(fr, fr0 | (S & ~vis0)) and np.array_equal(vis, vis0 | S)
            if len(ids) and n_bits > 1:
                vis, fr = vis0.copy(), fr0.copy()
                with pytest.raises(oracle_mod.OracleError) as ei:
                    oracle_mod.decompress_to_frontier(s, W, fr, vis, int(ids[-1]) - id_base, id_base=id_base)
                assert ei.value.code == oracle_mod.ERR_DST_TOO_SMALL
                assert np.array_equal(fr, fr0) and np.array_equal(vis, vis0)


def _pack_bits(bits):
    n = len(bits)
    words = (n + 31) // 32
    pad = np.zeros(words * 32, dtype=bool)
    pad[:n] = bits
    return np.packbits(pad.reshape(-1, 32), axis=1, bitorder="little").view(np.uint32).reshape(-1) if words else np.zeros(0, np.uint32)


def test_vbitmap_container(oracle_mod):
    """FORMAT.md §10: header typed by hand, the inner stream read back by the second
    witness, the minority / tie / not-smaller rules from closed forms, complement symmetry, identity round trip, rejects."""
    o = oracle_mod
    # a hand example: 1000 bits, set {3, 500, 999}: the three set bits are listed (kind 1)
    bits = np.zeros(1000, dtype=bool)
    bits[[3, 500, 999]] = True
    c = o.compress_vbitmap(_pack_bits(bits), 1000)
    inner = o.compress(np.array([3, 500, 999], dtype=np.uint32), 0)
    header = b"BFSV" + bytes([1, 32, 1, 0]) + (1000).to_bytes(8, "little") + (32 + len(inner)).to_bytes(8, "little") + (3).to_bytes(8, "little")
    assert c.tobytes() == header + inner.tobytes()
    assert witness.decode_stream(c[32:].tobytes(), 32) == [3, 500, 999]
    # the complement: the same three positions are now the CLEAR bits: kind 2, same stream
    c2 = o.compress_vbitmap(_pack_bits(~bits), 1000)
    assert c2[6] == 2 and c2[32:].tobytes() == inner.tobytes() and c2[:6].tobytes() == c[:6].tobytes() and c2[8:].tobytes() == c[8:].tobytes()
    assert np.array_equal(o.decompress_vbitmap(c2, 1000), _pack_bits(~bits))
    # closed forms: an empty stream is 48 bytes (32-byte header + the 16-byte directory of zero blocks)
    for n_bits in (4097, 1 << 16):
        z = o.compress_vbitmap(_pack_bits(np.zeros(n_bits, bool)), n_bits)
        f = o.compress_vbitmap(_pack_bits(np.ones(n_bits, bool)), n_bits)
        assert (z[6], len(z), f[6], len(f)) == (1, 80, 2, 80)
        assert int.from_bytes(z[24:32].tobytes(), "little") == 0
    # half of the bits set, even as one run (gaps of 1: b = 1, 32 bytes per 128 IDs = 2 bits per ID = 1 bit per vertex,
    # plus the directory): never smaller than the bitmap -> kind 0; the minority side decides from there on
    tie = np.zeros(1 << 14, dtype=bool)
    tie[:1 << 13] = True
    assert o.compress_vbitmap(_pack_bits(tie), 1 << 14)[6] == 0
    few = np.zeros(1 << 14, dtype=bool)
    few[:1 << 10] = True                                          # 1024 of 16384 set: listed; all but 1024 set: the clear ones
    assert o.compress_vbitmap(_pack_bits(few), 1 << 14)[6] == 1 and o.compress_vbitmap(_pack_bits(~few), 1 << 14)[6] == 2
    # not smaller than the bitmap itself -> kind 0, payload = the bitmap's bytes, bits >= n_bits written as 0
    rng = np.random.default_rng(3)
    half = rng.random(5000) < 0.5
    bm = _pack_bits(half)
    dirty = bm.copy()
    dirty[-1] |= np.uint32(0xFFFFFFFF) << np.uint32(5000 % 32)    # garbage beyond n_bits in the caller's last word
    k0 = o.compress_vbitmap(dirty, 5000)
    raw = (4 * len(bm) + 15) // 16 * 16
    assert k0[6] == 0 and len(k0) == 32 + raw == o.vbitmap_bound(5000)
    assert k0[32:32 + 4 * len(bm)].tobytes() == bm.tobytes() and not k0[32 + 4 * len(bm):].any()
    assert k0.tobytes() == o.compress_vbitmap(bm, 5000).tobytes()
    # tiny bitmaps: the 48-byte empty stream is never smaller than <= 48 bytes of bitmap
    for n_bits in (0, 1, 31, 32, 33, 384):
        t = o.compress_vbitmap(_pack_bits(np.zeros(n_bits, bool)), n_bits)
        assert t[6] == 0 and len(t) == o.vbitmap_bound(n_bits)
    assert o.compress_vbitmap(_pack_bits(np.zeros(385, bool)), 385)[6] == 1     # 64 bytes of bitmap: the empty stream wins
    # identity and the size bound over densities, both rules
    for n_bits in (1, 127, 128, 4096, 70001):
        for dens in (0.0, 0.001, 0.05, 0.3, 0.5, 0.7, 0.95, 0.999, 1.0):
            b = rng.random(n_bits) < dens
            for codec in (o.CODEC_PFOR, o.CODEC_BP128):
                cc = o.compress_vbitmap(_pack_bits(b), n_bits, codec)
                assert len(cc) <= o.vbitmap_bound(n_bits) and len(cc) % 16 == 0
                assert int.from_bytes(cc[16:24].tobytes(), "little") == len(cc)
                assert np.array_equal(o.decompress_vbitmap(cc, n_bits), _pack_bits(b))
                k = int(b.sum())
                if cc[6]:
                    assert cc[6] == (1 if k <= n_bits - k else 2) and int.from_bytes(cc[24:32].tobytes(), "little") == min(k, n_bits - k)
    # rejects
    def rc_of(buf, n_bits):
        try:
            o.decompress_vbitmap(buf, n_bits)
            return 0
        except o.OracleError as e:
            return e.code
    assert rc_of(c, 1000) == 0
    for pos, val in ((0, ord("X")), (4, 2), (5, 64), (6, 3), (7, 1), (24, 4)):      # magic, version, width, kind, byte 7, n_listed
        bad = c.copy()
        bad[pos] = val
        assert rc_of(bad, 1000) == 3, pos
    assert rc_of(c, 1001) == 2 and rc_of(c[:-16], 1000) == 3
    bad = k0.copy()
    bad[32 + 5000 // 8] |= 1 << 7                                  # a pad bit of a kind-0 payload
    assert rc_of(bad, 5000) == 3
    far = o.compress_vbitmap(_pack_bits(bits), 1000).copy()        # claim fewer bits than the listed IDs need
    far[8:16] = np.frombuffer((600).to_bytes(8, "little"), dtype=np.uint8)
    assert rc_of(far, 600) == 3
